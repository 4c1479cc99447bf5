// nrr_match_common.cuh -- device helpers shared by the matching kernels (nrr_match.cu, nrr_match_pair.cu):
// mbarrier / TMA PTX wrappers, reductions, the FP64 two-pass NCC used for photo-finish re-scoring, result
// write-back.  CUDA path only; nothing here is shared with oracle/.
#pragma once

#include <cuda.h>
#include <math.h>
#include <stdint.h>

#include "nrr_internal.cuh"

namespace nrr {
namespace {

__host__ __device__ inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// ------------------------------------------------------------------------------------------ PTX helpers
#ifdef NRR_EMUL      // CPU test build (tests/cuda_emul): same interface, emulated barrier and copy engine
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)(uintptr_t)p; }
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) { emul::mbar_init(bar, count); }
__device__ __forceinline__ void mbar_fence_init() {}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes) { emul::mbar_arrive_expect_tx(bar, bytes); }
__device__ __forceinline__ bool mbar_try_wait(uint64_t *bar, uint32_t parity) { return emul::mbar_try_wait(bar, parity); }
__device__ __forceinline__ bool mbar_wait(uint64_t *bar, uint32_t parity, const unsigned int *)
{
    for (int spin = 0; spin < 3; ++spin)
        if (mbar_try_wait(bar, parity)) return true;
    emul::mbar_timeout();
    return false;
}
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *map, int x, int y, int z, uint64_t *bar)
{
    emul::tma_load_3d(dst, map, x, y, z, bar);
}
#else
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ uint64_t global_timer_ns()
{
    uint64_t t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
// Bounded wait: a mis-programmed copy must neither hang the GPU nor fault it.  Returns false when the barrier has
// not completed after kMbarTimeoutNs of wall time (bounded by time, not by polls: time-slicing, a debugger or a long
// TMA queue must not fire it on a healthy copy); the caller then reports NRR_E_DEVICE through the sticky error
// flag and leaves the kernel in an orderly way -- no __trap(), no Xid.
// Fail fast once one CTA has given up: a wait that has lasted kMbarPeekNs (a healthy copy lands in microseconds) also
// looks at the sticky error flag, so the CTAs behind the first time-out leave after a millisecond each instead of
// holding the GPU for the full bound round after round (19,757 CTAs of config 4 would be 134 rounds x 4 s).
constexpr uint64_t kMbarTimeoutNs = 4000000000ull;
constexpr uint64_t kMbarPeekNs = 1000000ull;
__device__ __forceinline__ bool mbar_wait(uint64_t *bar, uint32_t parity, const unsigned int *err_flag)
{
    if (mbar_try_wait(bar, parity)) return true;
    const uint64_t t0 = global_timer_ns();
    while (!mbar_try_wait(bar, parity)) {
        const uint64_t dt = global_timer_ns() - t0;
        if (dt <= kMbarPeekNs) continue;
        if (dt > kMbarTimeoutNs) return false;
        if (err_flag && (*(const volatile unsigned int *)err_flag & 2u /* kErrStaging */)) return false;
    }
    return true;
}
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *map, int x, int y, int z, uint64_t *bar)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(x), "r"(y), "r"(z), "r"(smem_u32(bar))
        : "memory");
}

#endif

// ------------------------------------------------------------------------------------------ reductions
__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;   // butterfly: every lane holds the same bits
}

// Sum over the CTA in a fixed order; s_red needs 32 doubles. All threads must call.
__device__ double block_sum(double v, double *s_red)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = (blockDim.x + 31) >> 5;
    v = warp_sum(v);
    __syncthreads();
    if (lane == 0) s_red[warp] = v;
    __syncthreads();
    double t = 0.0;
    for (int w = 0; w < nwarp; ++w) t += s_red[w];
    return t;
}

__device__ __forceinline__ bool better(float v, int i, float bv, int bi) { return v > bv || (v == bv && i < bi); }
__device__ __forceinline__ bool better64(double v, int i, double bv, int bi) { return v > bv || (v == bv && i < bi); }

// CTA-wide arg-max with the lowest-index tie rule. Result valid in every thread. s_v/s_i: 32 entries each.
__device__ void block_argmax(float &v, int &i, float *s_v, int *s_i)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const float ov = __shfl_xor_sync(0xffffffffu, v, o);
        const int oi = __shfl_xor_sync(0xffffffffu, i, o);
        if (better(ov, oi, v, i)) { v = ov; i = oi; }
    }
    __syncthreads();
    if (lane == 0) { s_v[warp] = v; s_i[warp] = i; }
    __syncthreads();
    v = s_v[0]; i = s_i[0];
    for (int w = 1; w < nwarp; ++w)
        if (better(s_v[w], s_i[w], v, i)) { v = s_v[w]; i = s_i[w]; }
}

// Two-pass FP64 NCC of the fixed block at origin o and the moving block at origin p, by one warp.
// The summation order depends only on the position inside the block, so equal contents give equal bits.
__device__ double ncc64_warp(const float *__restrict__ fixed, const float *__restrict__ moving, Int3 dims,
                             Int3 block, int ox, int oy, int oz, int px, int py, int pz)
{
    const int lane = threadIdx.x & 31;
    const int nvox = block.x * block.y * block.z;
    const int bxy = block.x * block.y;
    double sf = 0.0, sm = 0.0;
    for (int i = lane; i < nvox; i += 32) {
        const int z = i / bxy, r = i - z * bxy, y = r / block.x, x = r - y * block.x;
        sf += (double)__ldg(fixed + ((size_t)(oz + z) * dims.y + (oy + y)) * dims.x + ox + x);
        sm += (double)__ldg(moving + ((size_t)(pz + z) * dims.y + (py + y)) * dims.x + px + x);
    }
    const double mf = warp_sum(sf) / (double)nvox, mm = warp_sum(sm) / (double)nvox;
    double ssf = 0.0, ssm = 0.0, c = 0.0;
    for (int i = lane; i < nvox; i += 32) {
        const int z = i / bxy, r = i - z * bxy, y = r / block.x, x = r - y * block.x;
        const double df = (double)__ldg(fixed + ((size_t)(oz + z) * dims.y + (oy + y)) * dims.x + ox + x) - mf;
        const double dm = (double)__ldg(moving + ((size_t)(pz + z) * dims.y + (py + y)) * dims.x + px + x) - mm;
        ssf += df * df;
        ssm += dm * dm;
        c += df * dm;
    }
    ssf = warp_sum(ssf);
    ssm = warp_sum(ssm);
    c = warp_sum(c);
    return (ssf == 0.0 || ssm == 0.0) ? 0.0 : c / sqrt(ssf * ssm);
}

struct TieScratch {
    int count;            // near-tie candidates besides the FP32 best
    float best_v;
    int best_i;
    double w_v[32];
    int w_i[32];
};

// Re-scores the FP32 best and the listed near-ties in FP64 and writes the result. All threads call;
// s_list holds ts->count candidate indices. (wx, wy) = candidates per row / rows per plane.
__device__ void rescore_and_write(const float *fixed, const float *moving, Int3 dims, Int3 block, Int3 window,
                                  int ox, int oy, int oz, const int *s_list, TieScratch *ts, int b,
                                  int *out_disp, float *out_ncc)
{
    const int wx = 2 * window.x + 1, wy = 2 * window.y + 1;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = (blockDim.x + 31) >> 5;
    const int entries = ts->count + 1;
    double bv = -INFINITY;
    int bi = 0x7fffffff;
    for (int e = warp; e < entries; e += nwarp) {
        const int idx = e == 0 ? ts->best_i : s_list[e - 1];
        const int dz = idx / (wx * wy) - window.z, r = idx % (wx * wy), dy = r / wx - window.y, dx = r % wx - window.x;
        const double v = ncc64_warp(fixed, moving, dims, block, ox, oy, oz, ox + dx, oy + dy, oz + dz);
        if (better64(v, idx, bv, bi)) { bv = v; bi = idx; }
    }
    if (lane == 0) { ts->w_v[warp] = bv; ts->w_i[warp] = bi; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 0; w < nwarp; ++w)
            if (better64(ts->w_v[w], ts->w_i[w], bv, bi)) { bv = ts->w_v[w]; bi = ts->w_i[w]; }
        const int dz = bi / (wx * wy) - window.z, r = bi % (wx * wy), dy = r / wx - window.y, dx = r % wx - window.x;
        out_disp[3 * (size_t)b + 0] = dx;
        out_disp[3 * (size_t)b + 1] = dy;
        out_disp[3 * (size_t)b + 2] = dz;
        out_ncc[b] = (float)bv;
    }
}

__device__ __forceinline__ void write_result(int idx, float v, Int3 window, int b, int *out_disp, float *out_ncc)
{
    const int wx = 2 * window.x + 1, wy = 2 * window.y + 1;
    const int dz = idx / (wx * wy) - window.z, r = idx % (wx * wy), dy = r / wx - window.y, dx = r % wx - window.x;
    out_disp[3 * (size_t)b + 0] = dx;
    out_disp[3 * (size_t)b + 1] = dy;
    out_disp[3 * (size_t)b + 2] = dz;
    out_ncc[b] = v;
}

__device__ __forceinline__ bool block_in_volume(Int3 dims, Int3 block, int ox, int oy, int oz)
{
    return ox >= 0 && oy >= 0 && oz >= 0 && ox + block.x <= dims.x && oy + block.y <= dims.y && oz + block.z <= dims.z;
}

// Sticky device-side error flag bits (read and cleared by nrr_bm_check_async_error)
constexpr unsigned int kErrBounds = 1u;      // a supplied block leaves the volume       -> NRR_E_BOUNDS
constexpr unsigned int kErrStaging = 2u;     // a staged (TMA / bulk) copy did not land  -> NRR_E_DEVICE

__device__ void write_error_result(int b, int *out_disp, float *out_ncc, unsigned int *err_flag, unsigned int bit)
{
    if (threadIdx.x == 0) {
        out_disp[3 * (size_t)b + 0] = 0;
        out_disp[3 * (size_t)b + 1] = 0;
        out_disp[3 * (size_t)b + 2] = 0;
        out_ncc[b] = __int_as_float(0x7fc00000);
        atomicOr(err_flag, bit);
    }
}
__device__ __forceinline__ void write_bounds_error(int b, int *out_disp, float *out_ncc, unsigned int *err_flag)
{
    write_error_result(b, out_disp, out_ncc, err_flag, kErrBounds);
}

// row[k] = row[k + S] for k < UX, in place, one thread per row: whole row to registers, then vector stores.
template <int S, int UX, int PITCH>
__device__ __forceinline__ void shift_row_left(float *row)
{
    constexpr int NL = (UX + S + 3) / 4;        // vectors holding the shifted source
    constexpr int NS = (UX + 3) / 4;            // vectors written
    static_assert(NL * 4 <= PITCH, "row pitch too small for the alignment slack");
    float t[NL * 4 + 4];
#pragma unroll
    for (int q = 0; q < NL; ++q) {
        const float4 v = *reinterpret_cast<const float4 *>(row + 4 * q);
        t[4 * q + 0] = v.x; t[4 * q + 1] = v.y; t[4 * q + 2] = v.z; t[4 * q + 3] = v.w;
    }
#pragma unroll
    for (int k = NL * 4; k < NL * 4 + 4; ++k) t[k] = 0.f;
#pragma unroll
    for (int q = 0; q < NS; ++q)
        *reinterpret_cast<float4 *>(row + 4 * q) = make_float4(t[4 * q + S], t[4 * q + 1 + S], t[4 * q + 2 + S], t[4 * q + 3 + S]);
}

constexpr int pitch_for(int ux)
{
    int p = (ux + 3 + 3) / 4 * 4;               // room for the 0..3 floats of TMA alignment slack
    return ((p / 4) % 2 == 0) ? p + 4 : p;      // 4 * odd
}

}  // namespace

// host side (defined in nrr_match.cu)
bool make_volume_map(CUtensorMap *map, const float *vol, Int3 dims, int bx, int by, int bz);
bool tma_eligible(Int3 dims, const void *moving, int box_z);

}  // namespace nrr
