// nrr_boxstat.cu -- per-candidate normalisers of the moving volume.
//
// For every block ORIGIN p of the moving volume whose block fits, the sum of squared deviations
//     SS(p) = sum m^2 - (sum m)^2 / N     over the B voxels of the block at p
// is formed from separable sliding box sums in IEEE double (m^2 of an fp32 is exact in double; the
// sums-form loses < 1e-13 relative here) and stored as inv_sd[p] = 1/sqrt(SS(p)) in fp32.  NCC's
// denominator then costs the matching kernel one multiply per candidate, and "only the
// cross term is recomputed" per candidate (BASELINE.json north_star).
//
// Zero-variance blocks (reading Q12: NCC := 0) get inv_sd = 0.  In the sums-form an exactly constant block
// can leave a rounding residue, so SS <= 2^-40 * sum m^2 counts as zero.
//
// One CTA owns a TX x TY tile of origins in (x,y) and marches over a chunk of z: each input plane is staged
// in shared memory with its (B-1) halo, reduced along x, then along y, and enters a running z-sum through a
// ring of the last Bz plane sums.  The kernel is bound by L2/HBM traffic (4 B read + 4 B written per voxel)
// and its double-precision adds, not by the FP32 pipe.
#include "nrr_internal.cuh"

namespace nrr {

namespace {

constexpr int TX = 32, TY = 8, ZCHUNK = 32;
constexpr int kThreads = TX * TY;

__global__ void __launch_bounds__(kThreads)
boxstat_kernel(const float *__restrict__ vol, Int3 dims, Int3 block, float *__restrict__ inv_sd)
{
    NRR_DYN_SMEM(s_dyn);
    // carve: row sums (double2) | ring (double2) | plane tile (float)
    const int HX = TX + block.x - 1, HY = TY + block.y - 1;
    double2 *s_row = (double2 *)s_dyn;                       // [HY][TX]
    double2 *s_ring = s_row + (size_t)HY * TX;               // [block.z][kThreads]
    float *s_plane = (float *)(s_ring + (size_t)block.z * kThreads);   // [HY][HX]

    const int tx = threadIdx.x % TX, ty = threadIdx.x / TX;
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY, z0 = blockIdx.z * ZCHUNK;
    const int nzo = dims.z - block.z + 1;                    // valid origins along z
    const int zo_end = min(z0 + ZCHUNK, nzo);                // exclusive
    const int zi_end = zo_end + block.z - 1;                 // exclusive input plane
    const double nvox = (double)((long long)block.x * block.y * block.z);
    const bool out_ok = (x0 + tx <= dims.x - block.x) && (y0 + ty <= dims.y - block.y);

    double run1 = 0.0, run2 = 0.0;
    for (int zi = z0; zi < zi_end; ++zi) {
        // stage the plane tile with halo (zero beyond the volume; those origins are never written)
        for (int i = threadIdx.x; i < HX * HY; i += kThreads) {
            const int lx = i % HX, ly = i / HX;
            const int gx = x0 + lx, gy = y0 + ly;
            s_plane[i] = (gx < dims.x && gy < dims.y) ? __ldg(vol + ((size_t)zi * dims.y + gy) * dims.x + gx) : 0.f;
        }
        __syncthreads();
        // x pass: sums of block.x consecutive voxels for every staged row
        for (int i = threadIdx.x; i < HY * TX; i += kThreads) {
            const int lx = i % TX, ly = i / TX;
            const float *p = s_plane + ly * HX + lx;
            double a = 0.0, b = 0.0;
            for (int k = 0; k < block.x; ++k) {
                const double v = (double)p[k];
                a += v;
                b = fma(v, v, b);
            }
            s_row[i] = make_double2(a, b);
        }
        __syncthreads();
        // y pass: this thread's column of block.y row sums -> plane sum
        double p1 = 0.0, p2 = 0.0;
        for (int k = 0; k < block.y; ++k) {
            const double2 r = s_row[(ty + k) * TX + tx];
            p1 += r.x;
            p2 += r.y;
        }
        // z: running sum over the last block.z planes
        const int slot = (zi - z0) % block.z;
        double2 *ring = s_ring + (size_t)slot * kThreads + threadIdx.x;
        if (zi - z0 >= block.z) {
            const double2 old = *ring;
            run1 -= old.x;
            run2 -= old.y;
        }
        run1 += p1;
        run2 += p2;
        *ring = make_double2(p1, p2);
        const int zo = zi - (block.z - 1);
        if (zo >= z0 && out_ok) {
            const double ss = run2 - run1 * run1 / nvox;
            float r = 0.f;
            if (ss > run2 * 9.094947017729282e-13 /* 2^-40 */) r = (float)(1.0 / sqrt(ss));
            inv_sd[((size_t)zo * dims.y + (y0 + ty)) * dims.x + (x0 + tx)] = r;
        }
        // s_plane is rewritten only after the next __syncthreads pair; s_row after the next x pass, which
        // sits behind the barrier that follows the next staging loop.
    }
}

}  // namespace

int boxstat_enqueue(const float *moving, Int3 dims, Int3 block, float *inv_sd, cudaStream_t stream)
{
    const int nxo = dims.x - block.x + 1, nyo = dims.y - block.y + 1, nzo = dims.z - block.z + 1;
    if (nxo < 1 || nyo < 1 || nzo < 1) return NRR_OK;
    const int HX = TX + block.x - 1, HY = TY + block.y - 1;
    const size_t smem = sizeof(double2) * ((size_t)HY * TX + (size_t)block.z * kThreads) + sizeof(float) * (size_t)HX * HY;
    if (smem > 200 * 1024) {
        set_error("block %dx%dx%d too large for the moving-volume statistics kernel", block.x, block.y, block.z);
        return NRR_E_SMEM;
    }
    if (smem > 48 * 1024)
        NRR_CUDA(cudaFuncSetAttribute(boxstat_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    dim3 grid((nxo + TX - 1) / TX, (nyo + TY - 1) / TY, (nzo + ZCHUNK - 1) / ZCHUNK);
    if (grid.y > 65535 || grid.z > 65535) {
        set_error("volume too large for the moving-volume statistics grid");
        return NRR_E_DIMS;
    }
    NRR_LAUNCH(boxstat_kernel, grid, kThreads, smem, stream, moving, dims, block, inv_sd);
    NRR_LAUNCH_CHECK("boxstat_kernel");
    return NRR_OK;
}

}  // namespace nrr
