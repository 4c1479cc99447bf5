// nrr_warp.cu -- warp of an image by a dense displacement field ("dense
// deformation field that defines transformation for each point in the image space"; reading Q21 of DESIGN.md):
//     out(p) = T[image](p + v(p)),  T = trilinear interpolation (x, then y, then z), sample clamped to the volume.
// One thread per output voxel, x fastest: the three field components and the output are read / written fully
// coalesced; the eight gathers of a warp fall into a few neighbouring rows of the image (L1/L2 hits for the
// smooth fields the method produces).  Bound: HBM, 4 B image + 12 B field + 4 B output per voxel.
//
// Precision: the sample position is split as p + floor(v) (integer arithmetic, exact) and v - floor(v) (exact in
// fp32), never formed as one fp32 number -- at x ~ 500 an fp32 position would carry 3e-5 voxels of rounding,
// i.e. 3e-3 intensity units on a steep edge.  The three interpolations run in fp32 (fmaf).
#include "nrr_internal.cuh"

namespace nrr {

namespace {

constexpr int kWarpThreads = 256;

// Splits the clamped sample coordinate pos + v into its lower voxel index, upper voxel index and fraction.
__device__ __forceinline__ void split_coord(int pos, float v, int n, int &i0, int &i1, float &t)
{
    const float fl = floorf(v);
    t = v - fl;                                   // exact
    // |v| beyond the volume clamps anyway: keep the integer part inside int range
    const float flc = fminf(fmaxf(fl, -2.0e9f), 2.0e9f);
    const long long s = (long long)pos + (long long)flc;
    if (s < 0) { i0 = 0; i1 = n > 1 ? 1 : 0; t = 0.f; }
    else if (s >= n - 1) { i0 = n - 1; i1 = n - 1; t = 0.f; }
    else { i0 = (int)s; i1 = i0 + 1; }
}

__global__ void __launch_bounds__(kWarpThreads)
warp_kernel(const float *__restrict__ image, Int3 dims, const float *__restrict__ field, float *__restrict__ out)
{
    const size_t nvox = (size_t)dims.x * dims.y * dims.z;
    const size_t p = (size_t)blockIdx.x * kWarpThreads + threadIdx.x;
    if (p >= nvox) return;
    const int x = (int)(p % dims.x);
    const int y = (int)((p / dims.x) % dims.y);
    const int z = (int)(p / ((size_t)dims.x * dims.y));
    int x0, x1, y0, y1, z0, z1;
    float tx, ty, tz;
    split_coord(x, __ldg(field + p), dims.x, x0, x1, tx);
    split_coord(y, __ldg(field + nvox + p), dims.y, y0, y1, ty);
    split_coord(z, __ldg(field + 2 * nvox + p), dims.z, z0, z1, tz);
    const float *r00 = image + ((size_t)z0 * dims.y + y0) * dims.x;
    const float *r01 = image + ((size_t)z0 * dims.y + y1) * dims.x;
    const float *r10 = image + ((size_t)z1 * dims.y + y0) * dims.x;
    const float *r11 = image + ((size_t)z1 * dims.y + y1) * dims.x;
    const float a00 = __ldg(r00 + x0), b00 = __ldg(r00 + x1);
    const float a01 = __ldg(r01 + x0), b01 = __ldg(r01 + x1);
    const float a10 = __ldg(r10 + x0), b10 = __ldg(r10 + x1);
    const float a11 = __ldg(r11 + x0), b11 = __ldg(r11 + x1);
    const float c00 = fmaf(tx, b00 - a00, a00), c01 = fmaf(tx, b01 - a01, a01);
    const float c10 = fmaf(tx, b10 - a10, a10), c11 = fmaf(tx, b11 - a11, a11);
    const float c0 = fmaf(ty, c01 - c00, c00), c1 = fmaf(ty, c11 - c10, c10);
    out[p] = fmaf(tz, c1 - c0, c0);
}

}  // namespace

int warp_enqueue(const float *image, Int3 dims, const float *field, float *out, cudaStream_t stream)
{
    const size_t nvox = (size_t)dims.x * dims.y * dims.z;
    const size_t ctas = (nvox + kWarpThreads - 1) / kWarpThreads;
    if (ctas > 0x7fffffffull) {
        set_error("volume too large for the warp grid");
        return NRR_E_DIMS;
    }
    NRR_LAUNCH(warp_kernel, (unsigned int)ctas, kWarpThreads, 0, stream, image, dims, field, out);
    NRR_LAUNCH_CHECK("warp_kernel");
    return NRR_OK;
}

}  // namespace nrr
