// nrr_match.cu -- exhaustive NCC block matching.
//
// One CTA per block.  NCC's numerator over the centred fixed block f' = f - fbar is
//     num(d) = sum_v f'(v) * m(o + d + v)                       (sum f' = 0, so no moving mean is needed)
// and NCC(d) = num(d) * inv_sd_m(o + d) * inv_sd_f, with inv_sd_m precomputed per block origin of the
// moving volume by nrr_boxstat.cu.  (PAPER.md:243-246 equation; listing PAPER.md:659-667.)
//
// FAST KERNEL (cubic block B in {5,7,9,11}, window (R,R,rz) with R in {3,5,7,9}):
//   M1  stage   : the union of the window's moving voxels arrives in shared memory by ONE TMA tensor copy
//                 (cp.async.bulk.tensor.3d; out-of-volume voxels are zero-filled by the hardware).  TMA needs
//                 a 16-byte aligned inner start coordinate (measured on B200: an unaligned x start raises an
//                 illegal-instruction fault), so the box starts at x rounded down to a multiple of 4 and each
//                 row is then shifted left by the 0..3 floats of slack, in place, with vector loads/stores.
//                 The union rows have a pitch of 4*odd floats and each z-plane holds W + 8k rows, so the
//                 LDS.128 row loads of a quarter-warp touch eight distinct 16-byte bank groups.
//   M3  cross   : one thread per candidate ROW (dy,dz): the W = 2R+1 candidates along x live in registers;
//                 per fixed-block row the thread loads B+W-1 moving floats (LDS.128) and B fixed floats
//                 (warp-broadcast LDS.128) and issues B*W FFMAs.
//   M4  argmax  : NCC in registers, lowest-linear-index tie rule, warp-shuffle + cross-warp reduction, then
//                 every candidate within kTieBand of the FP32 maximum is re-scored in FP64 (two-pass, from
//                 the raw voxels) and the decision is taken on the FP64 values.
//   M5  write   : out_disp, out_ncc.
// GENERIC KERNEL: any odd block / any window; fixed block in shared memory, moving voxels read through L1.
#include <cuda.h>
#include <math.h>
#include <string.h>

#include "nrr_match_common.cuh"

namespace nrr {

float g_tie_band = 1e-4f;     // FP32 candidates this close to the FP32 maximum are re-scored in FP64
int g_force_generic = 0;
int g_disable_tma = 0;
int g_force_rows = 0;          // != 0: skip the pair kernel (one candidate row per thread instead)

namespace {


// ------------------------------------------------------------------------------------------ fast kernel
template <int B, int R>
struct FastCfg {
    static constexpr int W = 2 * R + 1;                       // candidates per row; rows per z-plane of candidates
    static constexpr int UX = B + 2 * R;                      // union extent in x and y
    static constexpr int PITCH = pitch_for(UX);               // floats per staged row
    static constexpr int PROWS = W + 8 * ((B - 1 + 7) / 8);   // staged rows per z-plane (>= UX, == W mod 8)
    static constexpr int NV = (UX + 3) / 4;                   // LDS.128 per moving row
    static constexpr int FP = (B + 3) / 4 * 4;                // floats per staged fixed row
    static constexpr int NF = FP / 4;
    static constexpr int ROW_INSTR = B * W + NV + NF;
    static constexpr int UNROLL_VY = (B * ROW_INSTR * 16 <= 24 * 1024) ? B : ((24 * 1024) / (ROW_INSTR * 16) > 0 ? (24 * 1024) / (ROW_INSTR * 16) : 1);
    static_assert(PROWS >= UX, "plane rows must cover the union");
    static_assert(PITCH >= NV * 4, "row pitch must cover the vector loads");
};

struct FastSmem {      // tail of the dynamic shared memory, after the union and the fixed block
    uint64_t bar_union;
    double red[32];
    float am_v[32];
    int am_i[32];
    TieScratch ts;
    float isd_f;
    int stage_failed;
};


template <int B, int R>
__host__ __device__ inline size_t fast_union_bytes(int rz)
{
    using C = FastCfg<B, R>;
    return align_up(sizeof(float) * (size_t)(B + 2 * rz) * C::PROWS * C::PITCH, 128);
}
template <int B, int R>
__host__ __device__ inline size_t fast_fixed_bytes()
{
    using C = FastCfg<B, R>;
    return align_up(sizeof(float) * (size_t)B * B * C::FP, 128);
}
template <int B, int R>
inline size_t fast_smem_bytes(int rz)
{
    return fast_union_bytes<B, R>(rz) + fast_fixed_bytes<B, R>() + align_up(sizeof(FastSmem), 16) + 128;
}

constexpr int kFastMaxThreads = 512;

template <int B, int R>
__global__ void __launch_bounds__(kFastMaxThreads) match_rows_kernel(const __grid_constant__ CUtensorMap tm_moving, int use_tma,
                                  const float *__restrict__ fixed, const float *__restrict__ moving,
                                  const float *__restrict__ inv_sd, Int3 dims, const int *__restrict__ blocks,
                                  int rz, float tie_band, int *__restrict__ out_disp, float *__restrict__ out_ncc,
                                  unsigned int *err_flag, const unsigned int *__restrict__ n_dev)
{
    using C = FastCfg<B, R>;
    if (n_dev && blockIdx.x >= *n_dev) return;      // uniform: the launch was sized for an upper bound
    constexpr int W = C::W, PITCH = C::PITCH, PROWS = C::PROWS, FP = C::FP;
    NRR_DYN_SMEM(s_raw);
    unsigned char *s_base = s_raw + ((128u - (smem_u32(s_raw) & 127u)) & 127u);   // keeps the shared address space
    float *s_union = (float *)s_base;
    float *s_fixed = (float *)(s_base + fast_union_bytes<B, R>(rz));
    FastSmem *sm = (FastSmem *)((unsigned char *)s_fixed + fast_fixed_bytes<B, R>());

    const int b = blockIdx.x;
    const int tid = threadIdx.x;
    const Int3 block = {B, B, B};
    const Int3 window = {R, R, rz};
    const int ox = blocks[3 * (size_t)b + 0] - (B - 1) / 2;
    const int oy = blocks[3 * (size_t)b + 1] - (B - 1) / 2;
    const int oz = blocks[3 * (size_t)b + 2] - (B - 1) / 2;
    if (!block_in_volume(dims, block, ox, oy, oz)) {      // uniform over the CTA
        write_bounds_error(b, out_disp, out_ncc, err_flag);
        return;
    }
    const int WZ = 2 * rz + 1, UZ = B + 2 * rz;
    const int nrows = W * WZ;

    // ---- M1: stage the fixed block and the window union
    const int x0 = ox - R;
    const int x0a = x0 & ~3;                  // floor to a multiple of 4 (two's complement), TMA alignment
    const int xoff = x0 - x0a;                // 0..3 floats of slack at the start of every staged row
    if (use_tma) {
        if (tid == 0) {
            sm->stage_failed = 0;
            mbar_init(&sm->bar_union, 1);
            mbar_fence_init();
            mbar_arrive_expect_tx(&sm->bar_union, (uint32_t)(sizeof(float) * (size_t)UZ * PROWS * PITCH));
            tma_load_3d(s_union, &tm_moving, x0a, oy - R, oz - rz, &sm->bar_union);
        }
    } else {
        const int ux = C::UX;
        for (int i = tid; i < UZ * ux * ux; i += blockDim.x) {
            const int z = i / (ux * ux), r = i % (ux * ux), y = r / ux, x = r % ux;
            const int gx = x0 + x, gy = oy - R + y, gz = oz - rz + z;
            float v = 0.f;
            if (gx >= 0 && gx < dims.x && gy >= 0 && gy < dims.y && gz >= 0 && gz < dims.z)
                v = __ldg(moving + ((size_t)gz * dims.y + gy) * dims.x + gx);
            s_union[((size_t)z * PROWS + y) * PITCH + x] = v;
        }
    }
    for (int i = tid; i < B * B * B; i += blockDim.x) {
        const int z = i / (B * B), r = i % (B * B), y = r / B, x = r % B;
        s_fixed[(z * B + y) * FP + x] = __ldg(fixed + ((size_t)(oz + z) * dims.y + (oy + y)) * dims.x + ox + x);
    }
    __syncthreads();                          // fixed block staged; barrier initialisation visible

    // ---- centre the fixed block in place: mean and SS in FP64, f' stored in FP32
    {
        double s = 0.0;
        for (int i = tid; i < B * B * B; i += blockDim.x) {
            const int zy = i / B, x = i % B;
            s += (double)s_fixed[zy * FP + x];
        }
        const double mean = block_sum(s, sm->red) / (double)(B * B * B);
        double q = 0.0;
        for (int i = tid; i < B * B * B; i += blockDim.x) {
            const int zy = i / B, x = i % B;
            const double d = (double)s_fixed[zy * FP + x] - mean;
            s_fixed[zy * FP + x] = (float)d;
            q += d * d;
        }
        const double ssf = block_sum(q, sm->red);
        if (tid == 0) sm->isd_f = ssf == 0.0 ? 0.f : (float)(1.0 / sqrt(ssf));
        __syncthreads();
    }
    const float isd_f = sm->isd_f;

    // ---- this thread's candidate row (dyi, dzi); idle lanes shadow the last row
    const int t = tid < nrows ? tid : nrows - 1;
    const int dyi = t % W, dzi = t / W;
    const int py = oy + dyi - R, pz = oz + dzi - rz;
    const bool row_ok = tid < nrows && py >= 0 && py + B <= dims.y && pz >= 0 && pz + B <= dims.z;

    // per-candidate normalisers, fetched early so the loads fly during the main loop
    float isd[W];
#pragma unroll
    for (int j = 0; j < W; ++j) {
        const int px = ox + j - R;
        isd[j] = (row_ok && px >= 0 && px + B <= dims.x) ? __ldg(inv_sd + ((size_t)pz * dims.y + py) * dims.x + px) : -1.f;
    }

    if (use_tma) {
        if (!mbar_wait(&sm->bar_union, 0, err_flag)) sm->stage_failed = 1;
        if (xoff != 0) {                      // uniform over the CTA
            const int nstaged = UZ * C::UX;   // rows that are read later: (z, y < UX)
            for (int r = tid; r < nstaged; r += blockDim.x) {
                float *row = s_union + ((size_t)(r / C::UX) * PROWS + (r % C::UX)) * PITCH;
                if (xoff == 1) shift_row_left<1, C::UX, PITCH>(row);
                else if (xoff == 2) shift_row_left<2, C::UX, PITCH>(row);
                else shift_row_left<3, C::UX, PITCH>(row);
            }
        }
        __syncthreads();
        if (sm->stage_failed) {      // uniform: the copy did not land in time -- report, never fault (NRR_E_DEVICE)
            write_error_result(b, out_disp, out_ncc, err_flag, kErrStaging);
            return;
        }
    }

    // ---- M3: cross terms
    float acc[W];
#pragma unroll
    for (int j = 0; j < W; ++j) acc[j] = 0.f;
    const float *urow = s_union + ((size_t)dzi * PROWS + dyi) * PITCH;
#pragma unroll 1
    for (int vz = 0; vz < B; ++vz) {
        const float *up = urow + (size_t)vz * PROWS * PITCH;
        const float *fp = s_fixed + vz * B * FP;
#pragma unroll(C::UNROLL_VY)
        for (int vy = 0; vy < B; ++vy) {
            float m[C::NV * 4];
            float f[FP];
#pragma unroll
            for (int q = 0; q < C::NV; ++q) {
                const float4 v4 = *reinterpret_cast<const float4 *>(up + vy * PITCH + 4 * q);
                m[4 * q + 0] = v4.x; m[4 * q + 1] = v4.y; m[4 * q + 2] = v4.z; m[4 * q + 3] = v4.w;
            }
#pragma unroll
            for (int q = 0; q < C::NF; ++q) {
                const float4 v4 = *reinterpret_cast<const float4 *>(fp + vy * FP + 4 * q);
                f[4 * q + 0] = v4.x; f[4 * q + 1] = v4.y; f[4 * q + 2] = v4.z; f[4 * q + 3] = v4.w;
            }
#pragma unroll
            for (int vx = 0; vx < B; ++vx)
#pragma unroll
                for (int j = 0; j < W; ++j) acc[j] = fmaf(f[vx], m[j + vx], acc[j]);
        }
    }

    // ---- M4: NCC, arg-max with the lowest-index rule
    float bv = -INFINITY;
    int bi = 0x7fffffff;
#pragma unroll
    for (int j = 0; j < W; ++j) {
        acc[j] = acc[j] * isd[j] * isd_f;
        if (isd[j] >= 0.f && acc[j] > bv) { bv = acc[j]; bi = t * W + j; }
    }
    block_argmax(bv, bi, sm->am_v, sm->am_i);

    // near ties: the union is dead now, its storage becomes the list
    int *s_list = (int *)s_union;
    if (tid == 0) { sm->ts.count = 0; sm->ts.best_v = bv; sm->ts.best_i = bi; }
    __syncthreads();
    const float thr = bv - tie_band;
#pragma unroll
    for (int j = 0; j < W; ++j) {
        const int idx = t * W + j;
        if (isd[j] >= 0.f && acc[j] >= thr && idx != bi) s_list[atomicAdd(&sm->ts.count, 1)] = idx;
    }
    __syncthreads();
    if (sm->ts.count == 0) {
        if (tid == 0) write_result(bi, bv, window, b, out_disp, out_ncc);
        return;
    }
    rescore_and_write(fixed, moving, dims, block, window, ox, oy, oz, s_list, &sm->ts, b, out_disp, out_ncc);
}

// ------------------------------------------------------------------------------------------ generic kernel
struct GenericSmem {
    double red[32];
    float am_v[32];
    int am_i[32];
    TieScratch ts;
    float isd_f;
};

__global__ void __launch_bounds__(128)
match_generic_kernel(const float *__restrict__ fixed, const float *__restrict__ moving,
                     const float *__restrict__ inv_sd, Int3 dims, const int *__restrict__ blocks, Int3 block,
                     Int3 window, float tie_band, int *__restrict__ out_disp, float *__restrict__ out_ncc,
                     unsigned int *err_flag, const unsigned int *__restrict__ n_dev)
{
    if (n_dev && blockIdx.x >= *n_dev) return;      // uniform: the launch was sized for an upper bound
    NRR_DYN_SMEM(s_raw);
    const int nvox = block.x * block.y * block.z;
    const int wx = 2 * window.x + 1, wy = 2 * window.y + 1, wz = 2 * window.z + 1;
    const int ncand = wx * wy * wz;
    GenericSmem *sm = (GenericSmem *)s_raw;
    float *s_f = (float *)(s_raw + align_up(sizeof(GenericSmem), 16));   // [nvox]
    float *s_ncc = s_f + nvox;                                           // [ncand]
    int *s_list = (int *)(s_ncc + ncand);                                // [ncand]

    const int b = blockIdx.x, tid = threadIdx.x;
    const int ox = blocks[3 * (size_t)b + 0] - (block.x - 1) / 2;
    const int oy = blocks[3 * (size_t)b + 1] - (block.y - 1) / 2;
    const int oz = blocks[3 * (size_t)b + 2] - (block.z - 1) / 2;
    if (!block_in_volume(dims, block, ox, oy, oz)) {
        write_bounds_error(b, out_disp, out_ncc, err_flag);
        return;
    }
    const int bxy = block.x * block.y;
    double s = 0.0;
    for (int i = tid; i < nvox; i += blockDim.x) {
        const int z = i / bxy, r = i - z * bxy, y = r / block.x, x = r - y * block.x;
        const float v = __ldg(fixed + ((size_t)(oz + z) * dims.y + (oy + y)) * dims.x + ox + x);
        s_f[i] = v;
        s += (double)v;
    }
    const double mean = block_sum(s, sm->red) / (double)nvox;
    double q = 0.0;
    for (int i = tid; i < nvox; i += blockDim.x) {
        const double d = (double)s_f[i] - mean;
        s_f[i] = (float)d;
        q += d * d;
    }
    const double ssf = block_sum(q, sm->red);
    if (tid == 0) sm->isd_f = ssf == 0.0 ? 0.f : (float)(1.0 / sqrt(ssf));
    __syncthreads();
    const float isd_f = sm->isd_f;

    float bv = -INFINITY;
    int bi = 0x7fffffff;
    for (int c = tid; c < ncand; c += blockDim.x) {
        const int dzi = c / (wx * wy), r = c - dzi * wx * wy, dyi = r / wx, dxi = r - dyi * wx;
        const int px = ox + dxi - window.x, py = oy + dyi - window.y, pz = oz + dzi - window.z;
        float v = -INFINITY;
        if (block_in_volume(dims, block, px, py, pz)) {
            float num = 0.f;
            int i = 0;
            for (int z = 0; z < block.z; ++z)
                for (int y = 0; y < block.y; ++y) {
                    const float *row = moving + ((size_t)(pz + z) * dims.y + (py + y)) * dims.x + px;
                    for (int x = 0; x < block.x; ++x, ++i) num = fmaf(s_f[i], __ldg(row + x), num);
                }
            v = num * __ldg(inv_sd + ((size_t)pz * dims.y + py) * dims.x + px) * isd_f;
            if (v > bv) { bv = v; bi = c; }
        }
        s_ncc[c] = v;
    }
    block_argmax(bv, bi, sm->am_v, sm->am_i);
    if (tid == 0) { sm->ts.count = 0; sm->ts.best_v = bv; sm->ts.best_i = bi; }
    __syncthreads();
    const float thr = bv - tie_band;
    for (int c = tid; c < ncand; c += blockDim.x)
        if (s_ncc[c] >= thr && c != bi) s_list[atomicAdd(&sm->ts.count, 1)] = c;
    __syncthreads();
    if (sm->ts.count == 0) {
        if (tid == 0) write_result(bi, bv, window, b, out_disp, out_ncc);
        return;
    }
    rescore_and_write(fixed, moving, dims, block, window, ox, oy, oz, s_list, &sm->ts, b, out_disp, out_ncc);
}

}  // namespace

// ------------------------------------------------------------------------------------------ host side
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled_fn()
{
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
        else
            (void)cudaGetLastError();
    }
    return fn;
}

bool make_volume_map(CUtensorMap *map, const float *vol, Int3 dims, int bx, int by, int bz)
{
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return false;
    cuuint64_t gdim[3] = {(cuuint64_t)dims.x, (cuuint64_t)dims.y, (cuuint64_t)dims.z};
    cuuint64_t gstr[2] = {(cuuint64_t)dims.x * 4, (cuuint64_t)dims.x * dims.y * 4};
    cuuint32_t box[3] = {(cuuint32_t)bx, (cuuint32_t)by, (cuuint32_t)bz};
    cuuint32_t estr[3] = {1, 1, 1};
    return fn(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void *)vol, gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
              CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

bool tma_eligible(Int3 dims, const void *moving, int box_z)
{
    if (g_disable_tma) return false;
    if (dims.x % 4 != 0) return false;                                   // global strides must be multiples of 16 B
    if ((uintptr_t)moving & 15) return false;
    if (box_z > 256) return false;
    return encode_tiled_fn() != nullptr;
}

namespace {

template <int B, int R>
int launch_fast(const MatchCall &c, MatchPlan *plan_only)
{
    using C = FastCfg<B, R>;
    const Int3 dims = c.dims;
    const float *moving = c.moving;
    const int rz = c.window.z, n = c.n;
    cudaStream_t stream = c.stream;
    const int nrows = C::W * (2 * rz + 1);
    const int threads = (nrows + 31) / 32 * 32;
    const size_t smem = fast_smem_bytes<B, R>(rz);
    const bool tma = tma_eligible(dims, moving, B + 2 * rz);
    if (plan_only) {
        plan_only->fast = 1;
        plan_only->threads = threads;
        plan_only->smem_bytes = (int)smem;
        plan_only->tma = tma ? 1 : 0;
        return NRR_OK;
    }
    CUtensorMap tm_m;
    memset(&tm_m, 0, sizeof(tm_m));
    int use_tma = 0;
    if (tma && make_volume_map(&tm_m, moving, dims, C::PITCH, C::PROWS, B + 2 * rz)) use_tma = 1;
    auto kern = match_rows_kernel<B, R>;
    static int configured_smem[kMaxDevices] = {};     // per instantiation and device
    int &conf = configured_smem[current_device()];
    if ((int)smem > conf) {
        NRR_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        conf = (int)smem;
    }
    profile_begin(2, stream);
    NRR_LAUNCH(kern, n, threads, smem, stream, tm_m, use_tma, c.fixed, moving, c.inv_sd, dims, c.blocks, rz, g_tie_band,
               c.out_disp, c.out_ncc, c.err_flag, c.n_dev);
    profile_end(2, stream);
    NRR_LAUNCH_CHECK("match_rows_kernel");
    return NRR_OK;
}

constexpr size_t kMaxSmem = 227 * 1024;

template <int B>
int dispatch_r(const MatchCall &c, MatchPlan *plan_only, bool *handled)
{
    const int r = c.window.x, rz = c.window.z;
    *handled = true;
#define NRR_CASE(RR)                                                                                              \
    case RR:                                                                                                      \
        if (FastCfg<B, RR>::W * (2 * rz + 1) <= kFastMaxThreads && fast_smem_bytes<B, RR>(rz) <= kMaxSmem)                   \
            return launch_fast<B, RR>(c, plan_only);                                                              \
        break;
    switch (r) {
        NRR_CASE(3)
        NRR_CASE(5)
        NRR_CASE(7)
        NRR_CASE(9)
    default:
        break;
    }
#undef NRR_CASE
    *handled = false;
    return NRR_OK;
}

int dispatch(const MatchCall &c, MatchPlan *plan_only)
{
    const Int3 block = c.block, window = c.window;
    const int n = c.n;
    cudaStream_t stream = c.stream;
    const long long ncand = (long long)(2 * window.x + 1) * (2 * window.y + 1) * (2 * window.z + 1);
    if (plan_only) plan_only->candidates = (int)(ncand > 0x7fffffff ? 0x7fffffff : ncand);
    bool handled = false;
    if (plan_only) plan_only->blocks_per_cta = 1;
    if (!g_force_generic && !g_force_rows) {
        const int rc = match_pair_dispatch(c, plan_only, &handled);
        if (rc != NRR_OK || handled) return rc;
    }
    if (c.phase == kMatchPrepOnly) return NRR_OK;      // only the pair kernel keeps fixed-block records
    if (!g_force_generic && block.x == block.y && block.y == block.z && window.x == window.y) {
        int rc = NRR_OK;
        switch (block.x) {
        case 5: rc = dispatch_r<5>(c, plan_only, &handled); break;
        case 7: rc = dispatch_r<7>(c, plan_only, &handled); break;
        case 9: rc = dispatch_r<9>(c, plan_only, &handled); break;
        case 11: rc = dispatch_r<11>(c, plan_only, &handled); break;
        default: break;
        }
        if (handled) return rc;
    }
    // generic kernel
    const long long nvox = (long long)block.x * block.y * block.z;
    const size_t smem = align_up(sizeof(GenericSmem), 16) + sizeof(float) * (size_t)nvox + 2 * sizeof(float) * (size_t)ncand;
    if (ncand > (1ll << 26) || smem > kMaxSmem) {
        set_error("block %dx%dx%d with window +-(%d,%d,%d) needs %zu B of shared memory (limit %zu)", block.x, block.y,
                  block.z, window.x, window.y, window.z, smem, kMaxSmem);
        return NRR_E_SMEM;
    }
    if (plan_only) {
        plan_only->fast = 0;
        plan_only->threads = 128;
        plan_only->smem_bytes = (int)smem;
        plan_only->tma = 0;
        return NRR_OK;
    }
    static int configured_smem[kMaxDevices] = {};     // per device (0: the 48 KB default)
    int &conf = configured_smem[current_device()];
    if ((int)smem > 48 * 1024 && (int)smem > conf) {
        NRR_CUDA(cudaFuncSetAttribute(match_generic_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        conf = (int)smem;
    }
    profile_begin(2, stream);
    NRR_LAUNCH(match_generic_kernel, n, 128, smem, stream, c.fixed, c.moving, c.inv_sd, c.dims, c.blocks, block, window,
               g_tie_band, c.out_disp, c.out_ncc, c.err_flag, c.n_dev);
    profile_end(2, stream);
    NRR_LAUNCH_CHECK("match_generic_kernel");
    return NRR_OK;
}

}  // namespace

int match_plan(Int3 dims, Int3 block, Int3 window, const void *moving_ptr, const void *fixed_ptr, MatchPlan *plan, int n)
{
    MatchCall c;
    c.n = n;
    c.fixed = (const float *)fixed_ptr;
    c.moving = (const float *)moving_ptr;
    c.dims = dims; c.block = block; c.window = window;
    return dispatch(c, plan);
}

int match_enqueue(const MatchCall &c)
{
    if (c.n == 0) return NRR_OK;
    return dispatch(c, nullptr);
}

size_t match_records_bytes(Int3 block, Int3 window, int n)
{
    if (g_force_generic || g_force_rows) return 0;
    return match_pair_records_bytes(block, window, n);
}

}  // namespace nrr
