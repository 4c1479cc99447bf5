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

int g_boxstat_generic = 0;      // != 0: always use the generic (any block shape) kernel

namespace {

constexpr int TX = 32, TY = 8, ZCHUNK = 32;
constexpr int kThreads = TX * TY;

__global__ void __launch_bounds__(kThreads)
boxstat_kernel(const float *__restrict__ vol, Int3 dims, Int3 block, int zo_lo, int zo_hi, float *__restrict__ inv_sd)
{
    NRR_DYN_SMEM(s_dyn);
    // carve: row sums (double2) | ring (double2) | plane tile (float)
    const int HX = TX + block.x - 1, HY = TY + block.y - 1;
    double2 *s_row = (double2 *)s_dyn;                       // [HY][TX]
    double2 *s_ring = s_row + (size_t)HY * TX;               // [block.z][kThreads]
    float *s_plane = (float *)(s_ring + (size_t)block.z * kThreads);   // [HY][HX]

    const int tx = threadIdx.x % TX, ty = threadIdx.x / TX;
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY, z0 = zo_lo + blockIdx.z * ZCHUNK;
    const int zo_end = min(z0 + ZCHUNK, zo_hi);              // exclusive; zo_hi <= number of valid origins along z
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


// ------------------------------------------------------------------------------------------ sliding kernel
// Blocks B x B x bz with B in {5,7,9,11} (any bz).  One CTA owns a TX x TY tile of ORIGINS and marches over a chunk of z.
//   z : every thread owns NCOL input columns (x,y) of the haloed tile and keeps, per column, the running FP64
//       sums of m and m^2 over the last B planes (the plane that leaves the window is read again: an L2 hit);
//   x : the z-summed plane goes to shared memory; a thread per (row, 8 origins) slides the B-wide window;
//   y : a thread per (column, TY/2 origins) slides along y and writes inv_sd, coalesced along x.
// O(1) FP64 additions per voxel and axis; traffic: each input plane is read once per CTA column (halo
// (TX+B-1)(TY+B-1)/(TX TY)), each origin written once.
template <int B>
struct SlideCfg {
    static constexpr int NT = 256;
    static constexpr int TX = 64;
    static constexpr int TY = B <= 5 ? 18 : 14;      // 14 keeps <7> and <9> free of register spills (ptxas -v)
    static constexpr int HX = TX + B - 1, HY = TY + B - 1;
    static constexpr int NCOL = (HX * HY + NT - 1) / NT;
    static constexpr int ZP = HX | 1;            // pitch of s_z rows, in double2 (odd: conflict-free column walks)
    static constexpr int RP = HY | 1;            // pitch of s_row columns, in double2
    static constexpr int XS = 8;                 // origins per x-pass thread
    static constexpr int YS = TY / 2;            // origins per y-pass thread
    static constexpr size_t SMEM = sizeof(double2) * ((size_t)HY * ZP + (size_t)TX * RP);
    static_assert(HY * (TX / XS) <= NT && TX * 2 <= NT, "pass tasks must fit the CTA");
};

template <int B>
__global__ void __launch_bounds__(256, 2)
boxstat_slide_kernel(const float *__restrict__ vol, Int3 dims, int bz, int zo_lo, int zo_hi, int zchunk, float *__restrict__ inv_sd)
{
    using C = SlideCfg<B>;
    constexpr int TX = C::TX, TY = C::TY, HX = C::HX, HY = C::HY, NCOL = C::NCOL, ZP = C::ZP, RP = C::RP;
    NRR_DYN_SMEM(s_dyn);
    double2 *s_z = (double2 *)s_dyn;             // [HY][ZP]  z-window sums of the current plane
    double2 *s_row = s_z + (size_t)HY * ZP;      // [TX][RP]  x-window sums, transposed

    const int tid = threadIdx.x;
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY, z0 = zo_lo + blockIdx.z * zchunk;
    const int zo_end = min(z0 + zchunk, zo_hi);
    if (z0 >= zo_end) return;                    // uniform over the CTA
    const int zi_end = zo_end + bz - 1;
    const size_t plane = (size_t)dims.x * dims.y;
    const double nvox = (double)(B * B * bz);

    int gofs[NCOL], sidx[NCOL];                  // global offset inside a plane (-1: outside the volume), s_z slot (-1: none)
#pragma unroll
    for (int c = 0; c < NCOL; ++c) {
        const int i = tid + c * C::NT;
        const int ly = i / HX, lx = i - ly * HX;
        const int gx = x0 + lx, gy = y0 + ly;
        sidx[c] = i < HX * HY ? ly * ZP + lx : -1;
        gofs[c] = (i < HX * HY && gx < dims.x && gy < dims.y) ? gy * dims.x + gx : -1;
    }
    double z1[NCOL], z2[NCOL];
#pragma unroll
    for (int c = 0; c < NCOL; ++c) { z1[c] = 0.0; z2[c] = 0.0; }

    for (int zi = z0; zi < zi_end; ++zi) {
        {
            const bool emit = zi - z0 >= bz - 1; // uniform: the window is full, plane zo = zi - (bz-1) is due
            const bool drop = zi - z0 >= bz;     // uniform: plane zi - bz leaves the window (re-read: an L2 hit)
            float vn[NCOL], vl[NCOL];
#pragma unroll
            for (int c = 0; c < NCOL; ++c) {
                vn[c] = gofs[c] >= 0 ? __ldg(vol + (size_t)zi * plane + gofs[c]) : 0.f;
                vl[c] = (drop && gofs[c] >= 0) ? __ldg(vol + (size_t)(zi - bz) * plane + gofs[c]) : 0.f;
            }
#pragma unroll
            for (int c = 0; c < NCOL; ++c) {
                const double dn = (double)vn[c], dl = (double)vl[c];
                z1[c] += dn - dl;
                z2[c] = fma(dn, dn, z2[c]);
                z2[c] = fma(-dl, dl, z2[c]);
                if (emit && sidx[c] >= 0) s_z[sidx[c]] = make_double2(z1[c], z2[c]);
            }
            if (!emit) continue;
            __syncthreads();
            // x pass: thread = (row r, 8 consecutive origins), lanes walk r
            if (tid < HY * (TX / C::XS)) {
                const int r = tid % HY, xs = (tid / HY) * C::XS;
                const double2 *zr = s_z + (size_t)r * ZP + xs;
                double a = 0.0, b = 0.0;
#pragma unroll
                for (int j = 0; j < B; ++j) { a += zr[j].x; b += zr[j].y; }
                s_row[(size_t)xs * RP + r] = make_double2(a, b);
#pragma unroll
                for (int j = 1; j < C::XS; ++j) {
                    const double2 in = zr[j + B - 1], out = zr[j - 1];
                    a += in.x - out.x;
                    b += in.y - out.y;
                    s_row[(size_t)(xs + j) * RP + r] = make_double2(a, b);
                }
            }
            __syncthreads();
            // y pass: thread = (column x, TY/2 consecutive origins), lanes walk x; writes are coalesced along x
            if (tid < TX * 2) {
                const int x = tid % TX, ys = (tid / TX) * C::YS;
                const double2 *col = s_row + (size_t)x * RP + ys;
                const int gx = x0 + x, zo = zi - (bz - 1);
                const bool x_ok = gx <= dims.x - B;
                double a = 0.0, b = 0.0;
#pragma unroll
                for (int j = 0; j < B; ++j) { a += col[j].x; b += col[j].y; }
#pragma unroll
                for (int j = 0; j < C::YS; ++j) {
                    if (j > 0) {
                        const double2 in = col[j + B - 1], out = col[j - 1];
                        a += in.x - out.x;
                        b += in.y - out.y;
                    }
                    const int gy = y0 + ys + j;
                    if (x_ok && gy <= dims.y - B) {
                        const double ss = b - a * a / nvox;
                        float rr = 0.f;
                        if (ss > b * 9.094947017729282e-13 /* 2^-40 */) rr = rsqrtf((float)ss);
                        inv_sd[(size_t)zo * plane + (size_t)gy * dims.x + gx] = rr;
                    }
                }
            }
            // the next plane's s_z stores follow this thread's y pass; every x-pass read of s_z precedes the
            // barrier above, and the next x pass writes s_row only behind the next plane's first barrier
        }
    }
}

template <int B>
int launch_slide(const float *moving, Int3 dims, int bz, float *inv_sd, int zo_lo, int zo_hi, cudaStream_t stream)
{
    using C = SlideCfg<B>;
    const int nxo = dims.x - B + 1, nyo = dims.y - B + 1, nzo = zo_hi - zo_lo;
    const int gx = (nxo + C::TX - 1) / C::TX, gy = (nyo + C::TY - 1) / C::TY;
    // enough CTAs for two per SM; chunks of at least 2B planes keep the z halo below 50 %
    int zsplit = (2 * 148 + gx * gy - 1) / (gx * gy);
    const int max_split = (nzo + 2 * bz - 1) / (2 * bz);
    if (zsplit > max_split) zsplit = max_split;
    if (zsplit < 1) zsplit = 1;
    const int zchunk = (nzo + zsplit - 1) / zsplit;
    zsplit = (nzo + zchunk - 1) / zchunk;
    if (gy > 65535 || zsplit > 65535) {
        set_error("volume too large for the moving-volume statistics grid");
        return NRR_E_DIMS;
    }
    auto kern = boxstat_slide_kernel<B>;
    static bool configured[kMaxDevices] = {};     // per instantiation and device
    bool &conf = configured[current_device()];
    if (!conf) {
        NRR_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM));
        conf = true;
    }
    NRR_LAUNCH(kern, dim3(gx, gy, zsplit), C::NT, C::SMEM, stream, moving, dims, bz, zo_lo, zo_hi, zchunk, inv_sd);
    NRR_LAUNCH_CHECK("boxstat_slide_kernel");
    return NRR_OK;
}

}  // namespace

int boxstat_enqueue(const float *moving, Int3 dims, Int3 block, float *inv_sd, cudaStream_t stream)
{
    return boxstat_enqueue_range(moving, dims, block, inv_sd, 0, dims.z - block.z + 1, stream);
}

int boxstat_enqueue_range(const float *moving, Int3 dims, Int3 block, float *inv_sd, int zo_lo, int zo_hi, cudaStream_t stream)
{
    const int nxo = dims.x - block.x + 1, nyo = dims.y - block.y + 1;
    if (zo_lo < 0) zo_lo = 0;
    if (zo_hi > dims.z - block.z + 1) zo_hi = dims.z - block.z + 1;
    const int nzo = zo_hi - zo_lo;
    if (nxo < 1 || nyo < 1 || nzo < 1) return NRR_OK;
    if (!g_boxstat_generic && block.x == block.y) {      // in-plane square, any extent along z
        switch (block.x) {
        case 5: return launch_slide<5>(moving, dims, block.z, inv_sd, zo_lo, zo_hi, stream);
        case 7: return launch_slide<7>(moving, dims, block.z, inv_sd, zo_lo, zo_hi, stream);
        case 9: return launch_slide<9>(moving, dims, block.z, inv_sd, zo_lo, zo_hi, stream);
        case 11: return launch_slide<11>(moving, dims, block.z, inv_sd, zo_lo, zo_hi, stream);
        default: break;
        }
    }
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
    NRR_LAUNCH(boxstat_kernel, grid, kThreads, smem, stream, moving, dims, block, zo_lo, zo_hi, inv_sd);
    NRR_LAUNCH_CHECK("boxstat_kernel");
    return NRR_OK;
}

}  // namespace nrr
