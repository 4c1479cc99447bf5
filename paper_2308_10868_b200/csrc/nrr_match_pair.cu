// nrr_match_pair.cu -- the register-tiled matching kernel for blocks B x B x bz, B in {5,7,9,11} at compile time,
// bz (odd, <= 11) at run time.
//
// NCC's numerator over the centred fixed block f' = f - fbar is num(d) = sum_v f'(v) * m(o + d + v)
// (sum f' = 0, so the moving mean drops out); NCC(d) = num(d) * inv_sd_m(o + d) * inv_sd_f with inv_sd_m
// precomputed per block origin of the moving volume (nrr_boxstat.cu).  PAPER.md:243-246 (NCC equation),
// listing PAPER.md:659-667 (for each block, for each candidate in the window, similarity, maximum).
//
// Two kernels per nrr_bm_match call:
//
//  prep_kernel<B>      one warp per block: FP64 mean and sum of squares of the fixed block, then one RECORD per
//                      block in global scratch, laid out exactly as the matching kernel wants it in shared
//                      memory: the centred block f' as rows of FP floats, a PAIR TABLE holding, for the planes
//                      zr = 1..B-1, the interleaved pairs (f'[zr][vy][vx], f'[zr-1][vy][vx]), and a header
//                      with 1/sqrt(SS_f).  Blocks that leave the volume are flagged here.
//
//  match_pair_kernel<B,R>  one CTA per group of G consecutive blocks.
//    M1 stage   : one elected warp issues, per block, ONE TMA tensor copy of the window union of the moving
//                 volume (cp.async.bulk.tensor.3d, out-of-volume voxels zero-filled by the hardware) and one
//                 bulk copy of the G records; a single mbarrier collects the bytes.  TMA needs a 16-byte
//                 aligned inner start coordinate on B200 (an unaligned x start raises an illegal-instruction
//                 fault), so the box starts at x rounded down to a multiple of 4 and every staged row is
//                 shifted left in place by its block's 0..3 floats of slack.
//    M3 cross   : a thread owns TWO candidate rows that are adjacent in z, (dy, 2p) and (dy, 2p+1), W = 2R+1
//                 candidates each, as W packed accumulator pairs.  Every moving row it loads (LDS.128) feeds
//                 both rows: plane zr of the union meets fixed plane zr for the first row and zr-1 for the
//                 second, so one FFMA2 (fma.rn.f32x2: scalar moving voxel x pair of fixed voxels from the pair
//                 table) does two useful FMAs per issue slot and halves the shared-memory traffic per FMA.
//                 The two end planes touch one row only and use plain FFMA on one half of the pair.  The
//                 odd plane of candidates (dz = 2rz) is handled by separate warps whose threads own two rows
//                 adjacent in y, (dy, 2rz) and (dy+1, 2rz) (plain FFMA; one row per block stays alone), so that
//                 every warp of the CTA carries two candidate rows per lane.
//                 Which lane takes which (block, dy, p) comes from a host-built table that packs the tasks of
//                 the G blocks into full warps and keeps the LDS.128 of each quarter-warp on distinct banks.
//    M4 argmax  : NCC in registers; per-block maximum through a warp reduction and one 64-bit shared atomicMax
//                 on (ordered NCC bits, ~index), i.e. lowest linear candidate index among equal maxima; every
//                 candidate within tie_band of the FP32 maximum is re-scored in FP64 (two-pass, raw voxels)
//                 and the decision is taken on the FP64 values.
//    M5 write   : out_disp, out_ncc.
#include <cuda.h>
#include <math.h>
#include <string.h>

#include <map>
#include <mutex>
#include <vector>

#include "nrr_match_common.cuh"

namespace nrr {

extern float g_tie_band;
extern int g_disable_tma;
int g_pair_g = 0;             // experiment knob: force the number of blocks per CTA (0 = planner's choice)
int g_debug_tx_extra = 0;     // test hook: over-programs the staging barrier so that its wait must time out

namespace {

typedef unsigned long long u64;

constexpr int kGMax = 8;
constexpr int kPairMaxThreads = 512;

template <int B, int R>
struct PairCfg {
    static constexpr int W = 2 * R + 1;                 // candidates per row
    static constexpr int UX = B + 2 * R;                // union extent in x and y
    static constexpr int PITCH = pitch_for(UX);         // floats per staged row: 4 * odd, >= UX + 3
    static constexpr int NV = (UX + 3) / 4;             // LDS.128 per moving row
    static constexpr int FP = (B + 3) / 4 * 4;          // floats per row of the plain centred block
    static constexpr int NF = FP / 4;
    static constexpr int FPP = (2 * B + 3) / 4 * 4;     // floats per row of the pair table
    static constexpr int NFP = FPP / 4;
    static constexpr int HDR_FLOATS = 4;                // isd_f, valid, 0, 0
    // record of one block of B x B x bz voxels (in-plane edge B at compile time, bz at run time)
    __host__ __device__ static constexpr int plain_floats(int bz) { return bz * B * FP; }
    __host__ __device__ static constexpr int pair_floats(int bz) { return (bz - 1) * B * FPP; }
    __host__ __device__ static constexpr int rec_floats(int bz) { return plain_floats(bz) + pair_floats(bz) + HDR_FLOATS; }
    __host__ __device__ static constexpr int rec_bytes(int bz) { return rec_floats(bz) * 4; }      // multiple of 16
    static_assert(FP % 4 == 0 && FPP % 4 == 0 && HDR_FLOATS % 4 == 0, "records are moved by 16-byte bulk copies");
    static constexpr int B_ROW_BYTES = FP * 4;          // one staged row of the centred block
    static_assert(PITCH >= NV * 4, "row pitch must cover the vector loads");
};

struct PairCtrl {              // tail of the dynamic shared memory
    uint64_t bar;
    int bidx[kGMax];           // index of the block in the caller's list
    u64 best[kGMax];           // (ordered NCC bits << 32) | ~index
    int4 org[kGMax];           // block origin (x, y, z), w = 1 if the block is inside the volume
    int count[kGMax];          // near ties besides the FP32 best
    int stage_failed;          // a thread's bounded wait for the staged copies gave up
    TieScratch ts;
};

// ------------------------------------------------------------------------------------------ PTX helpers
#ifdef NRR_EMUL
__device__ __forceinline__ void bulk_load(void *dst, const void *src, uint32_t bytes, uint64_t *bar) { emul::bulk_load(dst, src, bytes, bar); }
__device__ __forceinline__ void fma2s(u64 &acc, float m, u64 f)
{
    float a[2], b[2];
    memcpy(a, &acc, 8);
    memcpy(b, &f, 8);
    a[0] = fmaf(m, b[0], a[0]);
    a[1] = fmaf(m, b[1], a[1]);
    memcpy(&acc, a, 8);
}
__device__ __forceinline__ void fma_lo(u64 &acc, float x, float y)
{
    float a[2];
    memcpy(a, &acc, 8);
    a[0] = fmaf(x, y, a[0]);
    memcpy(&acc, a, 8);
}
__device__ __forceinline__ void fma_hi(u64 &acc, float x, float y)
{
    float a[2];
    memcpy(a, &acc, 8);
    a[1] = fmaf(x, y, a[1]);
    memcpy(&acc, a, 8);
}
#else
__device__ __forceinline__ void bulk_load(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
// (acc.lo, acc.hi) += m * (f.lo, f.hi): SASS FFMA2 with a scalar-broadcast operand
__device__ __forceinline__ void fma2s(u64 &acc, float m, u64 f)
{
    u64 mm;
    asm("mov.b64 %0, {%1, %1};" : "=l"(mm) : "f"(m));
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc) : "l"(mm), "l"(f));
}
__device__ __forceinline__ void fma_lo(u64 &acc, float a, float b)
{
    asm("{\n\t.reg .f32 lo, hi;\n\tmov.b64 {lo, hi}, %0;\n\tfma.rn.f32 lo, %1, %2, lo;\n\tmov.b64 %0, {lo, hi};\n\t}"
        : "+l"(acc) : "f"(a), "f"(b));
}
__device__ __forceinline__ void fma_hi(u64 &acc, float a, float b)
{
    asm("{\n\t.reg .f32 lo, hi;\n\tmov.b64 {lo, hi}, %0;\n\tfma.rn.f32 hi, %1, %2, hi;\n\tmov.b64 %0, {lo, hi};\n\t}"
        : "+l"(acc) : "f"(a), "f"(b));
}
#endif
__device__ __forceinline__ uint32_t order_bits(float v)      // monotone float -> unsigned, never 0 for |v| <= 1
{
    const uint32_t b = __float_as_uint(v + 0.f);              // -0 -> +0
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ float unorder_bits(uint32_t k)
{
    return __uint_as_float((k & 0x80000000u) ? (k & 0x7fffffffu) : ~k);
}

// ------------------------------------------------------------------------------------------ prep kernel
constexpr int kPrepWarps = 4;
constexpr int kMaxBZ = 11;          // largest block extent along z the pair kernel takes

template <int B, int R>
__global__ void __launch_bounds__(kPrepWarps * 32)
prep_kernel(const float *__restrict__ fixed, Int3 dims, const int *__restrict__ blocks, int n, int bz,
            const unsigned int *__restrict__ n_dev, float *__restrict__ records)
{
    if (n_dev) n = min(n, (int)*n_dev);               // the launch was sized for an upper bound
    using C = PairCfg<B, R>;
    const int NVOX = B * B * bz;
    const int REC_FLOATS = C::rec_floats(bz), PLAIN_FLOATS = C::plain_floats(bz), PAIR_FLOATS = C::pair_floats(bz);
    __shared__ float s_f[kPrepWarps][B * B * kMaxBZ];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int b = blockIdx.x * kPrepWarps + warp;
    if (b >= n) return;
    float *rec = records + (size_t)b * REC_FLOATS;
    float *hdr = rec + PLAIN_FLOATS + PAIR_FLOATS;
    const int ox = blocks[3 * (size_t)b + 0] - (B - 1) / 2;
    const int oy = blocks[3 * (size_t)b + 1] - (B - 1) / 2;
    const int oz = blocks[3 * (size_t)b + 2] - (bz - 1) / 2;
    if (!block_in_volume(dims, Int3{B, B, bz}, ox, oy, oz)) {      // uniform over the warp; the matching kernel reports it
        for (int i = lane; i < REC_FLOATS; i += 32) rec[i] = 0.f;      // header: isd_f = 0, valid = 0
        return;
    }
    float *f = s_f[warp];
    double s = 0.0;
    for (int i = lane; i < NVOX; i += 32) {
        const int z = i / (B * B), r = i % (B * B), y = r / B, x = r % B;
        const float v = __ldg(fixed + ((size_t)(oz + z) * dims.y + (oy + y)) * dims.x + ox + x);
        f[i] = v;
        s += (double)v;
    }
    const double mean = warp_sum(s) / (double)NVOX;
    double q = 0.0;
    for (int i = lane; i < NVOX; i += 32) {
        const double d = (double)f[i] - mean;
        f[i] = (float)d;
        q += d * d;
    }
    const double ssf = warp_sum(q);
    __syncwarp();
    // plain centred block: rows of FP floats, zero padded
    for (int i = lane; i < PLAIN_FLOATS; i += 32) {
        const int zy = i / C::FP, x = i % C::FP;
        rec[i] = x < B ? f[zy * B + x] : 0.f;
    }
    // pair table: for zr = 1..B-1 and every (vy, vx): (f'[zr][vy][vx], f'[zr-1][vy][vx])
    float *pt = rec + PLAIN_FLOATS;
    for (int i = lane; i < PAIR_FLOATS; i += 32) {
        const int row = i / C::FPP, k = i % C::FPP;         // row = (zr-1)*B + vy
        const int zr = row / B + 1, vy = row % B, vx = k >> 1, h = k & 1;
        pt[i] = vx < B ? f[((zr - h) * B + vy) * B + vx] : 0.f;
    }
    if (lane == 0) {
        hdr[0] = ssf == 0.0 ? 0.f : (float)(1.0 / sqrt(ssf));
        hdr[1] = 1.f;
        hdr[2] = 0.f;
        hdr[3] = 0.f;
    }
}

// ------------------------------------------------------------------------------------------ main loops
template <int NV>
__device__ __forceinline__ void load_row(float (&m)[NV * 4], const float *p)
{
#pragma unroll
    for (int q = 0; q < NV; ++q) {
        const float4 v = *reinterpret_cast<const float4 *>(p + 4 * q);
        m[4 * q + 0] = v.x; m[4 * q + 1] = v.y; m[4 * q + 2] = v.z; m[4 * q + 3] = v.w;
    }
}

// Two candidate rows per thread: row A at union plane offset 0, row B one plane further.
// urow = first moving row of A; rec = this block's record; ra/rb receive the raw numerators.
template <int B, int R>
__device__ __forceinline__ void pair_rows(const float *urow, const float *rec, int bz, float (&ra)[2 * R + 1], float (&rb)[2 * R + 1])
{
    using C = PairCfg<B, R>;
    constexpr int NVX = C::NV;
    constexpr int W = C::W, PITCH = C::PITCH, PLANE = C::UX * C::PITCH;
    u64 acc[W];
#pragma unroll
    for (int j = 0; j < W; ++j) acc[j] = 0ull;
    // plane 0: row A only, fixed plane 0
#pragma unroll 1
    for (int vy = 0; vy < B; ++vy) {
        float m[NVX * 4], f[C::FP];
        load_row<NVX>(m, urow + vy * PITCH);
        load_row<C::NF>(f, rec + vy * C::FP);
#pragma unroll
        for (int vx = 0; vx < B; ++vx)
#pragma unroll
            for (int j = 0; j < W; ++j) fma_lo(acc[j], f[vx], m[j + vx]);
    }
    // planes 1..bz-1: both rows, (f'[zr], f'[zr-1]) pairs
    const float *pt = rec + C::plain_floats(bz);
#pragma unroll 1
    for (int zr = 1; zr < bz; ++zr) {
        const float *up = urow + zr * PLANE;
        const float *fp = pt + (zr - 1) * B * C::FPP;
#pragma unroll 1
        for (int vy = 0; vy < B; ++vy) {
            float m[NVX * 4];
            u64 f[C::NFP * 2];
            load_row<NVX>(m, up + vy * PITCH);
#pragma unroll
            for (int q = 0; q < C::NFP; ++q) {
                const ulonglong2 v = *reinterpret_cast<const ulonglong2 *>(fp + vy * C::FPP + 4 * q);
                f[2 * q] = v.x; f[2 * q + 1] = v.y;
            }
#pragma unroll
            for (int vx = 0; vx < B; ++vx)
#pragma unroll
                for (int j = 0; j < W; ++j) fma2s(acc[j], m[j + vx], f[vx]);
        }
    }
    // plane bz: row B only, fixed plane bz-1
    {
        const float *up = urow + bz * PLANE;
        const float *fp = rec + (bz - 1) * B * C::FP;
#pragma unroll 1
        for (int vy = 0; vy < B; ++vy) {
            float m[NVX * 4], f[C::FP];
            load_row<NVX>(m, up + vy * PITCH);
            load_row<C::NF>(f, fp + vy * C::FP);
#pragma unroll
            for (int vx = 0; vx < B; ++vx)
#pragma unroll
                for (int j = 0; j < W; ++j) fma_hi(acc[j], f[vx], m[j + vx]);
        }
    }
#pragma unroll
    for (int j = 0; j < W; ++j) {
        ra[j] = __uint_as_float((uint32_t)(acc[j] & 0xffffffffull));
        rb[j] = __uint_as_float((uint32_t)(acc[j] >> 32));
    }
}

// The odd last plane of candidates (dz = 2 rz): two candidate rows adjacent in y per thread, (dy, 2rz) and (dy+1, 2rz).
// Row vy of the union meets fixed row vy for the first candidate row and vy-1 for the second, so every moving row
// loaded feeds both (plain FFMA on two sets of accumulators: a packed form would need a second pair table).  The
// first union row of a plane touches the first candidate row only, the row after the last the second only.  `second`
// is false for the one task per block whose row has no partner (W is odd): its rb is never used.
template <int B, int R>
__device__ __forceinline__ void ypair_rows(const float *urow, const float *rec, int bz, bool second, float (&ra)[2 * R + 1], float (&rb)[2 * R + 1])
{
    using C = PairCfg<B, R>;
    constexpr int NVX = C::NV;
    constexpr int W = C::W, PITCH = C::PITCH, PLANE = C::UX * C::PITCH;
#pragma unroll
    for (int j = 0; j < W; ++j) { ra[j] = 0.f; rb[j] = 0.f; }
#pragma unroll 1
    for (int vz = 0; vz < bz; ++vz) {
        const float *up = urow + vz * PLANE;
        const float *fp = rec + vz * B * C::FP;
        {   // union row 0: first candidate row only, fixed row 0
            float m[NVX * 4], f[C::FP];
            load_row<NVX>(m, up);
            load_row<C::NF>(f, fp);
#pragma unroll
            for (int vx = 0; vx < B; ++vx)
#pragma unroll
                for (int j = 0; j < W; ++j) ra[j] = fmaf(f[vx], m[j + vx], ra[j]);
        }
#pragma unroll 1
        for (int vy = 1; vy < B; ++vy) {
            float m[NVX * 4], fa[C::FP], fb[C::FP];
            load_row<NVX>(m, up + vy * PITCH);
            load_row<C::NF>(fa, fp + vy * C::FP);
            load_row<C::NF>(fb, fp + (vy - 1) * C::FP);
#pragma unroll
            for (int vx = 0; vx < B; ++vx)
#pragma unroll
                for (int j = 0; j < W; ++j) {
                    ra[j] = fmaf(fa[vx], m[j + vx], ra[j]);
                    rb[j] = fmaf(fb[vx], m[j + vx], rb[j]);
                }
        }
        if (second) {   // union row B: second candidate row only, fixed row B-1 (a row without a partner has no such union row)
            float m[NVX * 4], f[C::FP];
            load_row<NVX>(m, up + B * PITCH);
            load_row<C::NF>(f, fp + (B - 1) * C::FP);
#pragma unroll
            for (int vx = 0; vx < B; ++vx)
#pragma unroll
                for (int j = 0; j < W; ++j) rb[j] = fmaf(f[vx], m[j + vx], rb[j]);
        }
    }
}

// ------------------------------------------------------------------------------------------ the kernel
struct PairArgs {
    const float *fixed, *moving, *inv_sd, *records;
    const int *blocks;
    const uint32_t *task_tab;      // [threads]: valid << 31 | y-pair warp << 30 | g << 16 | dy << 8 | p (z-pair: plane pair; y-pair: 1 = the row dy+1 belongs to the task)
    const unsigned int *n_dev;     // nullable: the number of blocks is min(n, *n_dev)
    int *out_disp;
    float *out_ncc;
    Int3 dims;
    int n, rz, bz, G, n_pair_warps;
    int use_tma;                   // 0: the unions are staged with plain loads (volumes TMA cannot address)
    int union_stride;              // bytes between the unions of consecutive blocks of a CTA (multiple of 128)
    float tie_band;
    unsigned int *err_flag;        // sticky device flag (kErrStaging when the staged copies do not land)
    unsigned int debug_tx_extra;   // test hook (option "debug_expect_tx_extra"): bytes added to the expected copy size
};

template <int B, int R>
__global__ void __launch_bounds__(kPairMaxThreads, 1)
match_pair_kernel(const __grid_constant__ CUtensorMap tm_moving, const PairArgs a)
{
    using C = PairCfg<B, R>;
    constexpr int W = C::W, PITCH = C::PITCH, UX = C::UX, PLANE = C::UX * C::PITCH;
    NRR_DYN_SMEM(s_raw);
    unsigned char *s_base = s_raw + ((128u - (smem_u32(s_raw) & 127u)) & 127u);
    unsigned char *s_unions = s_base;
    float *s_recs = (float *)(s_base + (size_t)a.G * a.union_stride);
    const int bz = a.bz, REC_FLOATS = C::rec_floats(bz);
    PairCtrl *ctrl = (PairCtrl *)((unsigned char *)s_recs + (size_t)a.G * REC_FLOATS * 4);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n = a.n_dev ? min(a.n, (int)*a.n_dev) : a.n;
    const int b0 = blockIdx.x * a.G;
    if (b0 >= n) return;                               // uniform: the launch was sized for an upper bound
    const int gact = min(a.G, n - b0);
    const int rz = a.rz, WZ = 2 * rz + 1, UZ = bz + 2 * rz;
    const Int3 dims = a.dims;
    const uint32_t union_bytes = (uint32_t)(sizeof(float) * UZ * UX * PITCH);

    // ---- M1: stage. Warp 0: lane g owns block b0 + g.
    if (warp == 0) {
        if (lane == 0) {
            ctrl->stage_failed = 0;
            mbar_init(&ctrl->bar, 1);
            mbar_fence_init();
        }
        int ox = 0, oy = 0, oz = 0, ok = 0, bi = 0;
        if (lane < gact) {
            bi = b0 + lane;
            ox = a.blocks[3 * (size_t)bi + 0] - (B - 1) / 2;
            oy = a.blocks[3 * (size_t)bi + 1] - (B - 1) / 2;
            oz = a.blocks[3 * (size_t)bi + 2] - (bz - 1) / 2;
            ok = block_in_volume(dims, Int3{B, B, bz}, ox, oy, oz) ? 1 : 0;
        }
        if (lane < kGMax) {
            ctrl->bidx[lane] = bi;
            ctrl->org[lane] = make_int4(ox, oy, oz, ok);
            ctrl->best[lane] = 0ull;
            ctrl->count[lane] = 0;
        }
        const unsigned okmask = __ballot_sync(0xffffffffu, ok);
        // The lane that initialised the barrier also programs it and issues every copy (the order the round-1 kernel
        // ran on hardware: init, fence, expect_tx, copies, all by one thread); the other lanes only hand over their
        // block's origin.  The copy instructions take warp-uniform operands anyway.
        if (lane == 0)
            mbar_arrive_expect_tx(&ctrl->bar, (a.use_tma ? (uint32_t)__popc(okmask) * union_bytes : 0u) + (uint32_t)gact * REC_FLOATS * 4u + a.debug_tx_extra);
        for (int gg = 0; gg < gact; ++gg) {
            const int gx = __shfl_sync(0xffffffffu, ox, gg), gy = __shfl_sync(0xffffffffu, oy, gg), gz = __shfl_sync(0xffffffffu, oz, gg);
            if (lane == 0 && a.use_tma && ((okmask >> gg) & 1u))
                tma_load_3d(s_unions + (size_t)gg * a.union_stride, &tm_moving, (gx - R) & ~3, gy - R, gz - rz, &ctrl->bar);
        }
        if (lane == 0) bulk_load(s_recs, a.records + (size_t)b0 * REC_FLOATS, (uint32_t)gact * REC_FLOATS * 4u, &ctrl->bar);
    }
    // this lane's task
    const uint32_t task = a.task_tab[tid];
    const int g = (task >> 16) & 0xff, dyi = (task >> 8) & 0xff, p = task & 0xff;
    const bool is_pair = !((task >> 30) & 1);          // uniform over the warp
    const int dzA = is_pair ? 2 * p : WZ - 1;
    __syncthreads();                                   // org[] and the barrier are visible
    const int4 org = ctrl->org[g < gact ? g : 0];
    const bool active = (task >> 31) && g < gact && org.w;

    if (!a.use_tma) {      // plain-load staging straight to the final position (no alignment slack to undo)
        const int per_block = UZ * UX * UX;
        for (int i = tid; i < gact * per_block; i += blockDim.x) {
            const int gg = i / per_block, r = i - gg * per_block;
            const int4 o = ctrl->org[gg];
            if (!o.w) continue;
            const int zz = r / (UX * UX), yy = (r / UX) % UX, xx = r % UX;
            const int gx = o.x - R + xx, gy = o.y - R + yy, gz = o.z - rz + zz;
            float v = 0.f;
            if (gx >= 0 && gx < dims.x && gy >= 0 && gy < dims.y && gz >= 0 && gz < dims.z)
                v = __ldg(a.moving + ((size_t)gz * dims.y + gy) * dims.x + gx);
            ((float *)(s_unions + (size_t)gg * a.union_stride))[((size_t)zz * UX + yy) * PITCH + xx] = v;
        }
    }
    if (!mbar_wait(&ctrl->bar, 0, a.err_flag)) ctrl->stage_failed = 1;
    // ---- undo the TMA alignment slack: shift every staged row left by its block's 0..3 floats
    if (a.use_tma) {
        const int rows_per_block = UZ * UX;
        for (int r = tid; r < gact * rows_per_block; r += blockDim.x) {
            const int gg = r / rows_per_block, rr = r - gg * rows_per_block;
            const int4 o = ctrl->org[gg];
            const int xoff = (o.x - R) & 3;
            float *row = (float *)(s_unions + (size_t)gg * a.union_stride) + (size_t)rr * PITCH;
            if (!o.w || xoff == 0) continue;
            if (xoff == 1) shift_row_left<1, UX, PITCH>(row);
            else if (xoff == 2) shift_row_left<2, UX, PITCH>(row);
            else shift_row_left<3, UX, PITCH>(row);
        }
    }
    __syncthreads();
    if (ctrl->stage_failed) {      // uniform: the copies did not land in time -- report, never fault (NRR_E_DEVICE)
        for (int gg = 0; gg < gact; ++gg)
            if (ctrl->org[gg].w) write_error_result(ctrl->bidx[gg], a.out_disp, a.out_ncc, a.err_flag, kErrStaging);
        return;
    }

    // ---- M3: cross terms
    float ra[W], rb[W];
    const float *urow = (const float *)(s_unions + (size_t)g * a.union_stride) + (size_t)dzA * PLANE + dyi * PITCH;
    const float *rec = s_recs + (size_t)g * REC_FLOATS;
    // second candidate row of the task: one plane further (z-pair) or one row further (y-pair, unless the row is alone)
    const bool has_b = is_pair || p != 0;
    const int dyB = is_pair ? dyi : dyi + 1, dzB = is_pair ? dzA + 1 : dzA;
    if (active) {
        if (is_pair) pair_rows<B, R>(urow, rec, bz, ra, rb);
        else ypair_rows<B, R>(urow, rec, bz, has_b, ra, rb);
    }

    // ---- M4: NCC and the per-block arg-max
    float bv = -INFINITY;
    int bi = 0x7fffffff;
    if (active) {
        const float isd_f = rec[REC_FLOATS - C::HDR_FLOATS];
        const int py = org.y + dyi - R;
        const bool y_ok = py >= 0 && py + B <= dims.y;
        const int jlo = max(0, R - org.x), jhi = min(W - 1, dims.x - B - org.x + R);      // valid j range
        {
            const int pz = org.z + dzA - rz;
            const bool row_ok = y_ok && pz >= 0 && pz + bz <= dims.z;
            const float *ip = a.inv_sd + ((size_t)pz * dims.y + py) * dims.x + org.x - R;
#pragma unroll
            for (int j = 0; j < W; ++j) {
                const bool ok = row_ok && j >= jlo && j <= jhi;
                const float v = ok ? ra[j] * __ldg(ip + j) * isd_f : -INFINITY;
                ra[j] = v;
                if (v > bv) { bv = v; bi = (dzA * W + dyi) * W + j; }
            }
        }
        if (has_b) {
            const int pyb = org.y + dyB - R, pz = org.z + dzB - rz;
            const bool row_ok = pyb >= 0 && pyb + B <= dims.y && pz >= 0 && pz + bz <= dims.z;
            const float *ip = a.inv_sd + ((size_t)pz * dims.y + pyb) * dims.x + org.x - R;
#pragma unroll
            for (int j = 0; j < W; ++j) {
                const bool ok = row_ok && j >= jlo && j <= jhi;
                const float v = ok ? rb[j] * __ldg(ip + j) * isd_f : -INFINITY;
                rb[j] = v;
                if (v > bv) { bv = v; bi = (dzB * W + dyB) * W + j; }
            }
        }
    }
    {
        const bool have = bi != 0x7fffffff;
        const uint32_t khi = have ? order_bits(bv) : 0u, klo = have ? 0xffffffffu - (uint32_t)bi : 0u;
        const int gq = active ? g : 0x7fffffff;
        const int gmin = __reduce_min_sync(0xffffffffu, gq);
        const int gmax = __reduce_max_sync(0xffffffffu, active ? g : -1);
        for (int gg = gmin; gg <= gmax; ++gg) {          // warp-uniform bounds; empty when no lane is active
            const uint32_t mh = __reduce_max_sync(0xffffffffu, (active && g == gg) ? khi : 0u);
            const uint32_t ml = __reduce_max_sync(0xffffffffu, (active && g == gg && khi == mh) ? klo : 0u);
            if (lane == 0 && mh) atomicMax(&ctrl->best[gg], ((u64)mh << 32) | ml);
        }
    }
    __syncthreads();

    // ---- near ties: the unions are dead now, their storage holds the per-block lists
    if (active) {
        const u64 best = ctrl->best[g];
        const float thr = unorder_bits((uint32_t)(best >> 32)) - a.tie_band;
        const int big = (int)(0xffffffffu - (uint32_t)best);
        int *s_list = (int *)(s_unions + (size_t)g * a.union_stride);
#pragma unroll
        for (int j = 0; j < W; ++j) {
            const int idx = (dzA * W + dyi) * W + j;
            if (ra[j] >= thr && idx != big) s_list[atomicAdd(&ctrl->count[g], 1)] = idx;
        }
        if (has_b) {
#pragma unroll
            for (int j = 0; j < W; ++j) {
                const int idx = (dzB * W + dyB) * W + j;
                if (rb[j] >= thr && idx != big) s_list[atomicAdd(&ctrl->count[g], 1)] = idx;
            }
        }
    }
    __syncthreads();

    // ---- M5: write, with the FP64 photo finish where needed
    const Int3 block = {B, B, bz}, window = {R, R, rz};
    for (int gg = 0; gg < gact; ++gg) {
        const int4 o = ctrl->org[gg];
        if (!o.w) {                                      // the block leaves the volume: NaN + sticky flag (NRR_E_BOUNDS)
            write_bounds_error(ctrl->bidx[gg], a.out_disp, a.out_ncc, a.err_flag);
            continue;
        }
        const u64 best = ctrl->best[gg];
        const int big = (int)(0xffffffffu - (uint32_t)best);
        const int cnt = ctrl->count[gg];
        if (cnt == 0) {
            if (tid == 0) write_result(big, unorder_bits((uint32_t)(best >> 32)), window, ctrl->bidx[gg], a.out_disp, a.out_ncc);
            continue;
        }
        if (tid == 0) { ctrl->ts.count = cnt; ctrl->ts.best_i = big; }
        __syncthreads();
        rescore_and_write(a.fixed, a.moving, dims, block, window, o.x, o.y, o.z,
                          (const int *)(s_unions + (size_t)gg * a.union_stride), &ctrl->ts, ctrl->bidx[gg], a.out_disp, a.out_ncc);
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------ host side
struct PairGeom {
    int G, n_pair_warps, n_ypair_warps, threads;
    int pair_lanes_per_block, ypair_lanes_per_block;
    int union_stride;
    size_t smem;
    double efficiency;          // useful candidate rows / row slots of the busiest warp scheduler x 4
    int ctas_per_sm;
    int sched_max;              // row-units on the busiest scheduler (every warp carries two candidate rows per lane)
};

constexpr size_t kMaxSmemPerCta = 227 * 1024, kSmemPerSm = 228 * 1024;

template <int B, int R>
bool pair_geometry(int rz, int bz, int G, PairGeom *out)
{
    using C = PairCfg<B, R>;
    const int WZ = 2 * rz + 1, UZ = bz + 2 * rz, NP = WZ / 2;
    PairGeom g;
    g.G = G;
    g.pair_lanes_per_block = (C::W * NP + 7) / 8 * 8;
    g.ypair_lanes_per_block = ((C::W + 1) / 2 + 7) / 8 * 8;      // the last plane: (W-1)/2 pairs of rows and one row alone
    g.n_pair_warps = (G * g.pair_lanes_per_block + 31) / 32;
    g.n_ypair_warps = (G * g.ypair_lanes_per_block + 31) / 32;
    g.threads = (g.n_pair_warps + g.n_ypair_warps) * 32;
    g.union_stride = (int)align_up(sizeof(float) * (size_t)UZ * C::UX * C::PITCH, 128);
    g.smem = (size_t)G * g.union_stride + (size_t)G * C::rec_bytes(bz) + align_up(sizeof(PairCtrl), 16) + 128;
    if (g.threads > kPairMaxThreads || g.smem > kMaxSmemPerCta) return false;
    // The CTA is done when its busiest scheduler is (warp w issues from scheduler w % 4): efficiency counts the other
    // three schedulers' idle slots too.  Every warp carries two candidate rows per lane, so the busiest scheduler is the
    // one with the most warps.
    g.sched_max = 2 * ((g.n_pair_warps + g.n_ypair_warps + 3) / 4);
    g.efficiency = (double)G * C::W * WZ / 32.0 / (4.0 * g.sched_max);
    const int by_smem = (int)(kSmemPerSm / (g.smem + 1024));
    const int by_regs = 65536 / (g.threads * 112);
    g.ctas_per_sm = by_smem < by_regs ? by_smem : by_regs;
    if (g.ctas_per_sm < 1) g.ctas_per_sm = 1;
    *out = g;
    return true;
}

template <int B, int R>
bool pair_plan(int rz, int bz, PairGeom *best, int n = 0)
{
    // n > 0: the number of blocks of this launch.  CTAs are handed to SMs as they free up, so the launch ends when the
    // SM with the most CTAs does: with nCTA CTAs over the device's SMs the last round is only partly filled.  For small
    // block lists (config 2: 1,215 blocks) this term decides; for config 3 (2,053 CTAs over 148 SMs) it is 0.99.
    constexpr int kSms = 148;
    bool found = false;
    double best_score = 0.0;
    for (int G = 1; G <= kGMax; ++G) {
        if (g_pair_g && G != g_pair_g) continue;
        PairGeom g;
        if (!pair_geometry<B, R>(rz, bz, G, &g)) continue;
        // a lone CTA per SM cannot overlap its staging with another CTA's arithmetic
        double score = g.efficiency * (g.ctas_per_sm >= 2 ? 1.0 : 0.85);
        if (n > 0) {
            const int ctas = (n + G - 1) / G, rounds = (ctas + kSms - 1) / kSms;
            score *= (double)ctas / ((double)rounds * kSms);
        }
        // a larger group must be better by more than the model's resolution (1 %) to be taken
        if (!found || score > best_score * 1.01) { found = true; best_score = score; *best = g; }
    }
    return found;
}

// Lane -> task table.  Tasks of block g fill the lane segment [g*L, (g+1)*L); inside it they are grouped into
// quarter-warps so that the eight LDS.128 row addresses of a quarter fall on distinct 16-byte bank groups
// where the counts allow it (address of a task, in 16-byte units: P4*dy + PLANE4*dz, PLANE4 = P4*UX).
void place_tasks(std::vector<uint32_t> &tab, int lane0, int lanes, int g, const std::vector<int> &dy,
                 const std::vector<int> &p, const std::vector<int> &residue)
{
    // Every residue class hands one task to each quarter-group in index order (so a group never sees a residue
    // twice and never exceeds eight lanes); what a class has beyond the number of groups is overflow, and all
    // overflow is packed into the last groups that still have room: the unavoidable two-way conflicts end up in as
    // few quarter-warps as possible.
    const int ngroups = lanes / 8;
    std::vector<std::vector<int>> grp(ngroups);
    std::vector<int> overflow;
    for (int r = 0; r < 8; ++r) {
        int k = 0;
        for (size_t t = 0; t < dy.size(); ++t) {
            if (residue[t] != r) continue;
            if (k < ngroups) grp[k++].push_back((int)t);
            else overflow.push_back((int)t);
        }
    }
    for (int t : overflow) {
        int k = ngroups - 1;
        while (k >= 0 && grp[k].size() >= 8) --k;
        if (k >= 0) grp[k].push_back(t);      // k < 0 cannot happen: the segment holds at least dy.size() lanes
    }
    for (int k = 0; k < ngroups; ++k)
        for (size_t s = 0; s < grp[k].size(); ++s) {
            const int t = grp[k][s];
            tab[lane0 + 8 * k + (int)s] = 0x80000000u | ((uint32_t)g << 16) | ((uint32_t)dy[t] << 8) | (uint32_t)p[t];
        }
}

// Start rows of the y-pair tasks of the last candidate plane: rows are paired from 0 up to a pivot row that stays
// alone, then from pivot + 1 on, so that the starts run through even and then odd values -- with an odd row pitch (in
// 16-byte units) up to eight of them fall on distinct bank groups (W = 7, 11, 15: all of them).
inline void ypair_starts(int W, std::vector<int> *dy, std::vector<int> *has_partner)
{
    const int pivot = W - 1 < 6 ? W - 1 : 6;          // even, <= W - 1 (W is odd)
    for (int d = 0; d < pivot; d += 2) { dy->push_back(d); has_partner->push_back(1); }
    dy->push_back(pivot); has_partner->push_back(0);
    for (int d = pivot + 1; d + 1 < W; d += 2) { dy->push_back(d); has_partner->push_back(1); }
}

template <int B, int R>
std::vector<uint32_t> build_task_table(int rz, const PairGeom &g)
{
    using C = PairCfg<B, R>;
    const int WZ = 2 * rz + 1, NP = WZ / 2, P4 = C::PITCH / 4, PLANE4 = P4 * C::UX;
    std::vector<uint32_t> tab((size_t)g.threads, 0u);
    for (int blk = 0; blk < g.G; ++blk) {
        std::vector<int> dy, p, res;
        for (int pp = 0; pp < NP; ++pp)
            for (int d = 0; d < C::W; ++d) { dy.push_back(d); p.push_back(pp); res.push_back((P4 * d + PLANE4 * 2 * pp) & 7); }
        place_tasks(tab, blk * g.pair_lanes_per_block, g.pair_lanes_per_block, blk, dy, p, res);
        dy.clear(); p.clear(); res.clear();
        ypair_starts(C::W, &dy, &p);
        for (int d : dy) res.push_back((P4 * d + PLANE4 * (WZ - 1)) & 7);
        place_tasks(tab, g.n_pair_warps * 32 + blk * g.ypair_lanes_per_block, g.ypair_lanes_per_block, blk, dy, p, res);
    }
    for (int w = g.n_pair_warps; w < g.n_pair_warps + g.n_ypair_warps; ++w)
        for (int l = 0; l < 32; ++l) tab[(size_t)w * 32 + l] |= 0x40000000u;      // role bit, uniform over the warp
    return tab;
}

std::mutex g_tab_mutex;
std::map<long long, uint32_t *> g_tab_cache;      // (device, B, R, rz, G) -> device table
std::map<long long, cudaEvent_t> g_tab_ready;     // ... and the event behind its upload

template <int B, int R>
int task_table_device(int rz, const PairGeom &g, cudaStream_t stream, const uint32_t **out)
{
    int dev = 0;
    NRR_CUDA(cudaGetDevice(&dev));
    const long long key = ((((long long)dev * 32 + B) * 32 + R) * 512 + rz) * 16 + g.G;      // the table does not depend on bz
    std::lock_guard<std::mutex> lock(g_tab_mutex);
    auto it = g_tab_cache.find(key);
    if (it != g_tab_cache.end()) {
        cudaEvent_t &ready = g_tab_ready[key];
        if (ready) {      // the upload may still be in flight on another stream
            if (cudaEventQuery(ready) == cudaSuccess) { cudaEventDestroy(ready); ready = nullptr; }
            else { (void)cudaGetLastError(); NRR_CUDA(cudaStreamWaitEvent(stream, ready, 0)); }
        }
        *out = it->second;
        return NRR_OK;
    }
    const std::vector<uint32_t> tab = build_task_table<B, R>(rz, g);
    // First use of this (device, shape): the table goes up from a pinned copy that lives as long as the cache entry,
    // in stream order -- no host synchronisation (nrr_bm_register promises none).  Later calls on OTHER streams may
    // race this first copy in principle; they are ordered by the event recorded behind it.
    uint32_t *d = nullptr, *h = nullptr;
    NRR_CUDA(cudaMalloc((void **)&d, tab.size() * sizeof(uint32_t)));
    NRR_CUDA(cudaMallocHost((void **)&h, tab.size() * sizeof(uint32_t)));
    memcpy(h, tab.data(), tab.size() * sizeof(uint32_t));
    NRR_CUDA(cudaMemcpyAsync(d, h, tab.size() * sizeof(uint32_t), cudaMemcpyHostToDevice, stream));
    cudaEvent_t ready = nullptr;
    NRR_CUDA(cudaEventCreateWithFlags(&ready, cudaEventDisableTiming));
    NRR_CUDA(cudaEventRecord(ready, stream));
    g_tab_ready[key] = ready;
    g_tab_cache[key] = d;
    *out = d;
    return NRR_OK;
}

template <int B, int R>
int launch_pair(const MatchCall &c, MatchPlan *plan_only, bool *handled)
{
    using C = PairCfg<B, R>;
    const Int3 dims = c.dims;
    const int rz = c.window.z, bz = c.block.z, n = c.n;
    cudaStream_t stream = c.stream;
    *handled = false;
    PairGeom g;
    if (bz < 1 || bz > kMaxBZ || !pair_plan<B, R>(rz, bz, &g, n)) return NRR_OK;
    if (plan_only) {
        *handled = true;
        plan_only->fast = 2;
        plan_only->threads = g.threads;
        plan_only->smem_bytes = (int)g.smem;
        plan_only->tma = (g_disable_tma || dims.x % 4 != 0 || bz + 2 * rz > 256) ? 0 : 1;      // what the shape alone decides
        plan_only->blocks_per_cta = g.G;
        return NRR_OK;
    }
    *handled = true;
    AsyncScratch rec_buf(stream);
    float *records = c.records;
    if (!records) {
        if (c.phase != kMatchBoth) { set_error("the matching phases run separately only on caller-kept records"); return NRR_E_ARG; }
        NRR_CUDA(rec_buf.alloc((size_t)n * C::rec_bytes(bz)));
        records = (float *)rec_buf.p;
    }
    if (c.phase != kMatchKernelOnly) {
        auto prep = prep_kernel<B, R>;
        profile_begin(3, stream);
        NRR_LAUNCH(prep, (n + kPrepWarps - 1) / kPrepWarps, kPrepWarps * 32, 0, stream, c.fixed, dims, c.blocks, n, bz, c.n_dev, records);
        profile_end(3, stream);
        NRR_LAUNCH_CHECK("prep_kernel");
        if (c.phase == kMatchPrepOnly) return NRR_OK;
    }
    // ---- what the copy engines need, checked on the host: a mis-programmed copy is refused here, never launched
    static_assert(C::PITCH % 4 == 0 && C::PITCH <= 256 && C::UX <= 256, "TMA box: inner extent a multiple of 16 bytes, extents <= 256");
    static_assert(C::rec_bytes(1) % 16 == 0 && (C::B_ROW_BYTES % 16) == 0, "bulk copies move multiples of 16 bytes");
    CUtensorMap tm_m;
    memset(&tm_m, 0, sizeof(tm_m));
    const int use_tma = tma_eligible(dims, c.moving, bz + 2 * rz) && make_volume_map(&tm_m, c.moving, dims, C::PITCH, C::UX, bz + 2 * rz);
    if (g.union_stride % 128 != 0 || ((size_t)g.G * g.union_stride) % 16 != 0 || ((uintptr_t)records & 15) != 0 ||
        C::rec_bytes(bz) % 16 != 0 || (size_t)g.union_stride < sizeof(float) * (size_t)(bz + 2 * rz) * C::UX * C::PITCH) {
        set_error("pair kernel: staging layout violates the copy engines' alignment rules (union stride %d, record %d B)",
                  g.union_stride, C::rec_bytes(bz));
        return NRR_E_ARG;
    }
    const uint32_t *tab = nullptr;
    int rc = task_table_device<B, R>(rz, g, stream, &tab);
    if (rc) return rc;
    auto kern = match_pair_kernel<B, R>;
    static size_t configured_smem[kMaxDevices] = {};     // per instantiation and device
    size_t &conf = configured_smem[current_device()];
    if (g.smem > conf) {
        NRR_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)g.smem));
        // two CTAs per SM only fit if the L1/shared split is at its shared-memory maximum
        NRR_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared));
        conf = g.smem;
    }
    PairArgs a;
    a.fixed = c.fixed; a.moving = c.moving; a.inv_sd = c.inv_sd; a.records = records; a.blocks = c.blocks; a.task_tab = tab;
    a.out_disp = c.out_disp; a.out_ncc = c.out_ncc; a.dims = dims; a.n = n; a.rz = rz; a.bz = bz; a.G = g.G; a.n_dev = c.n_dev;
    a.use_tma = use_tma;
    a.n_pair_warps = g.n_pair_warps; a.union_stride = g.union_stride; a.tie_band = g_tie_band;
    a.err_flag = c.err_flag; a.debug_tx_extra = (unsigned int)g_debug_tx_extra;
    profile_begin(2, stream);
    NRR_LAUNCH(kern, (n + g.G - 1) / g.G, g.threads, g.smem, stream, tm_m, a);
    profile_end(2, stream);
    NRR_LAUNCH_CHECK("match_pair_kernel");
    return NRR_OK;      // call scratch is released behind the kernels, in stream order
}

template <int B, int R>
size_t records_bytes_for(int rz, int bz, int n)
{
    PairGeom g;
    if (bz < 1 || bz > kMaxBZ || !pair_plan<B, R>(rz, bz, &g)) return 0;
    return (size_t)n * PairCfg<B, R>::rec_bytes(bz);
}

template <int B, int R>
int table_for(int rz, int bz, unsigned int *out, int capacity, int info[6])
{
    using C = PairCfg<B, R>;
    PairGeom g;
    if (bz < 1 || bz > kMaxBZ || !pair_plan<B, R>(rz, bz, &g)) return 0;
    info[0] = g.threads; info[1] = g.G; info[2] = C::PITCH; info[3] = C::UX; info[4] = g.union_stride; info[5] = (int)g.smem;
    if (capacity < g.threads) return -g.threads;
    const std::vector<uint32_t> tab = build_task_table<B, R>(rz, g);
    for (int i = 0; i < g.threads; ++i) out[i] = tab[(size_t)i];
    return g.threads;
}

}  // namespace

// The lane -> task table of the pair kernel for (block, window): returns the number of words written (threads per
// CTA), 0 if the pair kernel has no plan for this shape, -needed if `capacity` is too small.
int match_pair_table(Int3 block, Int3 window, unsigned int *out, int capacity, int info[6])
{
    if (!(block.x == block.y && window.x == window.y)) return 0;
#define NRR_PAIR(BB, RR) \
    if (block.x == BB && window.x == RR) return table_for<BB, RR>(window.z, block.z, out, capacity, info);
    NRR_PAIR(5, 3) NRR_PAIR(5, 5) NRR_PAIR(5, 7) NRR_PAIR(5, 9)
    NRR_PAIR(7, 3) NRR_PAIR(7, 5) NRR_PAIR(7, 7) NRR_PAIR(7, 9)
    NRR_PAIR(9, 3) NRR_PAIR(9, 5) NRR_PAIR(9, 7) NRR_PAIR(9, 9)
    NRR_PAIR(11, 3) NRR_PAIR(11, 5) NRR_PAIR(11, 7) NRR_PAIR(11, 9)
#undef NRR_PAIR
    return 0;
}

// Tries the pair kernel; *handled tells whether it took the call (blocks B x B x bz with B in 5/7/9/11 and any odd
// bz <= 11 -- thick-slice MRI wants e.g. 7 x 7 x 3 --, in-plane window 3/5/7/9 equal in x and y, any window in z).
int match_pair_dispatch(const MatchCall &c, MatchPlan *plan_only, bool *handled)
{
    *handled = false;
    const Int3 block = c.block, window = c.window;
    if (!(block.x == block.y && window.x == window.y)) return NRR_OK;
#define NRR_PAIR(BB, RR) \
    if (block.x == BB && window.x == RR) return launch_pair<BB, RR>(c, plan_only, handled);
    NRR_PAIR(5, 3) NRR_PAIR(5, 5) NRR_PAIR(5, 7) NRR_PAIR(5, 9)
    NRR_PAIR(7, 3) NRR_PAIR(7, 5) NRR_PAIR(7, 7) NRR_PAIR(7, 9)
    NRR_PAIR(9, 3) NRR_PAIR(9, 5) NRR_PAIR(9, 7) NRR_PAIR(9, 9)
    NRR_PAIR(11, 3) NRR_PAIR(11, 5) NRR_PAIR(11, 7) NRR_PAIR(11, 9)
#undef NRR_PAIR
    return NRR_OK;
}

size_t match_pair_records_bytes(Int3 block, Int3 window, int n)
{
    if (!(block.x == block.y && window.x == window.y)) return 0;
#define NRR_PAIR(BB, RR) \
    if (block.x == BB && window.x == RR) return records_bytes_for<BB, RR>(window.z, block.z, n);
    NRR_PAIR(5, 3) NRR_PAIR(5, 5) NRR_PAIR(5, 7) NRR_PAIR(5, 9)
    NRR_PAIR(7, 3) NRR_PAIR(7, 5) NRR_PAIR(7, 7) NRR_PAIR(7, 9)
    NRR_PAIR(9, 3) NRR_PAIR(9, 5) NRR_PAIR(9, 7) NRR_PAIR(9, 9)
    NRR_PAIR(11, 3) NRR_PAIR(11, 5) NRR_PAIR(11, 7) NRR_PAIR(11, 9)
#undef NRR_PAIR
    return 0;
}

}  // namespace nrr
