// nrr_fem.cu -- biomechanical regularisation of the sparse displacement field (include/nrr_bm.h
// "BIOMECHANICAL REGULARISATION").  PAPER.md:252-265 (section 3):
//
//        F_i <= K U_i ,      U_{i+1} <= [K + H^T S H]^-1 [H^T S D + F_i]
//
// K: stiffness of a linear elastic model on a tetrahedral mesh; H: interpolation from the mesh vertices to the block
// centres; S: confidence of the matches; D: the displacements nrr_bm_match returned.  "Both block matching and
// iterative estimation of displacements are time critical".
//
// The mesh is a regular grid of nodes whose cells are cut into the six Kuhn tetrahedra around the main diagonal
// (reading Q22: the paper's mesher is out of scope).  On such a mesh every operator is a 27-point stencil:
//   K        never assembled globally.  One 8 x 8 table of 3 x 3 blocks between the local vertices of a CELL (the sum of
//            its six constant-strain elements, K_ab = V (lambda g_a g_b^T + mu g_b g_a^T + mu (g_a . g_b) I)) is built
//            by fem_cell_kernel; K u at a node is the sum over its <= 8 cells of table blocks times neighbour values.
//   H^T S H  = W (x) I_3 with the scalar stencil W[node][27] = sum_k s_k w_k w_k^T; H^T S D = sum_k s_k w_k d_k^T:
//            one thread per block scatters its 4 x 4 + 4 x 3 contributions with FP64 atomics (fem_accumulate_kernel).
//   solve    Jacobi-preconditioned conjugate gradients in FP64, TWO kernels per iteration (the direction update
//            p = z + beta p_old is fused into the operator application: a neighbour's p is formed on the fly from z
//            and p_old, the directions ping-pong between two buffers), no host round trip inside an iteration: dot
//            products are reduced per CTA in a fixed order and finished by the last CTA to arrive (ticket), which
//            also updates alpha / beta / the convergence flag on the device.
#include <math.h>
#include <string.h>

#include "nrr_internal.cuh"

using namespace nrr;

namespace {

constexpr int kFemThreads = 128;
constexpr int kMaxParts = 4096;          // upper bound on CTAs of a PCG kernel (partial sums per CTA)

struct PcgState {
    double rz, pq, rr, bb, alpha, beta, tol2;
    int done, iters;
    unsigned int ticket;
};

struct FemGeom {
    Int3 dims, h, nn;       // volume, node spacing (voxels), nodes per axis
    int n;                  // nodes
};

__host__ __device__ inline int node_of(const FemGeom &g, int i, int j, int k) { return (k * g.nn.y + j) * g.nn.x + i; }

// Kuhn tetrahedron of permutation `perm` (axes in the order their unit steps are taken from vertex 0).
__constant__ int c_perm[6][3] = {{0, 1, 2}, {0, 2, 1}, {1, 0, 2}, {1, 2, 0}, {2, 0, 1}, {2, 1, 0}};

// ---- K: the cell table.  kcell[va][vb][3][3], local vertex index = dx + 2 dy + 4 dz.
__global__ void fem_cell_kernel(double hx, double hy, double hz, double lam, double mu, double *kcell)
{
    const int va = threadIdx.x >> 3, vb = threadIdx.x & 7;
    if (threadIdx.x >= 64) return;
    const double h[3] = {hx, hy, hz};
    const double vol = hx * hy * hz / 6.0;
    double acc[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
    for (int t = 0; t < 6; ++t) {
        // local vertices of this tetrahedron and the gradients of its barycentric coordinates
        int vert[4];
        double grad[4][3];
        for (int a = 0; a < 4; ++a) grad[a][0] = grad[a][1] = grad[a][2] = 0.0;
        int v = 0;
        vert[0] = 0;
        for (int s = 0; s < 3; ++s) {
            const int axis = c_perm[t][s];
            v |= 1 << axis;
            vert[s + 1] = v;
            grad[s][axis] -= 1.0 / h[axis];          // w_s = (coordinate s) - (coordinate s+1), w_0 = 1 - coordinate 1
            grad[s + 1][axis] += 1.0 / h[axis];
        }
        int ia = -1, ib = -1;
        for (int a = 0; a < 4; ++a) {
            if (vert[a] == va) ia = a;
            if (vert[a] == vb) ib = a;
        }
        if (ia < 0 || ib < 0) continue;
        const double *ga = grad[ia], *gb = grad[ib];
        const double dot = ga[0] * gb[0] + ga[1] * gb[1] + ga[2] * gb[2];
        for (int i = 0; i < 3; ++i)
            for (int j = 0; j < 3; ++j)
                acc[3 * i + j] += vol * (lam * ga[i] * gb[j] + mu * gb[i] * ga[j] + (i == j ? mu * dot : 0.0));
    }
    for (int e = 0; e < 9; ++e) kcell[(va * 8 + vb) * 9 + e] = acc[e];
}

// ---- point location (shared by the accumulation and the dense field): cell, Kuhn simplex, barycentric weights
__device__ __forceinline__ void locate(const FemGeom &g, double px, double py, double pz, int node[4], double w[4])
{
    const double p[3] = {px, py, pz};
    const int h[3] = {g.h.x, g.h.y, g.h.z}, nn[3] = {g.nn.x, g.nn.y, g.nn.z};
    int cell[3];
    double loc[3];
    for (int a = 0; a < 3; ++a) {
        int c = (int)floor(p[a] / (double)h[a]);
        c = c < 0 ? 0 : (c > nn[a] - 2 ? nn[a] - 2 : c);
        cell[a] = c;
        loc[a] = p[a] / (double)h[a] - (double)c;
    }
    // the permutation that sorts the local coordinates in descending order, ties to the lower axis
    int perm[3] = {0, 1, 2};
    for (int i = 1; i < 3; ++i)
        for (int j = i; j > 0 && loc[perm[j]] > loc[perm[j - 1]]; --j) { const int t = perm[j]; perm[j] = perm[j - 1]; perm[j - 1] = t; }
    int c[3] = {cell[0], cell[1], cell[2]};
    node[0] = node_of(g, c[0], c[1], c[2]);
    for (int s = 0; s < 3; ++s) {
        c[perm[s]] += 1;
        node[s + 1] = node_of(g, c[0], c[1], c[2]);
    }
    const double s0 = loc[perm[0]], s1 = loc[perm[1]], s2 = loc[perm[2]];
    w[0] = 1.0 - s0; w[1] = s0 - s1; w[2] = s1 - s2; w[3] = s2;
}

// ---- H^T S H and H^T S D: one thread per block
__global__ void __launch_bounds__(kFemThreads)
fem_accumulate_kernel(FemGeom g, const int *__restrict__ blocks, const int *__restrict__ disp, const float *__restrict__ ncc,
                      int n, double weight, double *wst, double *rhs0)
{
    const int b = blockIdx.x * kFemThreads + threadIdx.x;
    if (b >= n) return;
    const float c = ncc[b];
    if (!(c > 0.f)) return;                              // zero or negative confidence, NaN: no influence (reading Q24)
    const double s = weight * (double)c;
    int node[4];
    double w[4];
    locate(g, (double)blocks[3 * (size_t)b], (double)blocks[3 * (size_t)b + 1], (double)blocks[3 * (size_t)b + 2], node, w);
    const double d[3] = {(double)disp[3 * (size_t)b], (double)disp[3 * (size_t)b + 1], (double)disp[3 * (size_t)b + 2]};
    const int nx = g.nn.x, nxy = g.nn.x * g.nn.y;
    for (int a = 0; a < 4; ++a) {
        if (w[a] == 0.0) continue;
        const int ka = node[a] / nxy, ja = (node[a] - ka * nxy) / nx, ia = node[a] - ka * nxy - ja * nx;
        for (int e = 0; e < 4; ++e) {
            if (w[e] == 0.0) continue;
            const int ke = node[e] / nxy, je = (node[e] - ke * nxy) / nx, ie = node[e] - ke * nxy - je * nx;
            const int off = (ie - ia + 1) + 3 * (je - ja + 1) + 9 * (ke - ka + 1);
            atomicAdd(&wst[(size_t)node[a] * 27 + off], s * w[a] * w[e]);
        }
        for (int ax = 0; ax < 3; ++ax) atomicAdd(&rhs0[(size_t)node[a] * 3 + ax], s * w[a] * d[ax]);
    }
}

// ---- operator application at one node: y = [K u] (with_k) + [W u] (with_w)
// The operand is u, or u + beta * u2 when u2 != NULL (the search direction p = z + beta p_old formed on the fly, with the
// same explicitly fused operation wherever it is formed, so every thread sees the same bits for a given node).
__device__ __forceinline__ double operand(const double *__restrict__ u, const double *__restrict__ u2, double beta, size_t e)
{
    return u2 ? fma(beta, u2[e], u[e]) : u[e];
}

__device__ __forceinline__ void apply_node(const FemGeom &g, const double *__restrict__ kcell, const double *__restrict__ wst,
                                           const double *__restrict__ u, int i, int j, int k, bool with_k, bool with_w, double y[3],
                                           const double *__restrict__ u2 = nullptr, double beta = 0.0)
{
    y[0] = y[1] = y[2] = 0.0;
    if (with_k) {
        for (int cz = 0; cz < 2; ++cz)
            for (int cy = 0; cy < 2; ++cy)
                for (int cx = 0; cx < 2; ++cx) {
                    // the cell whose local vertex (cx, cy, cz) is this node
                    const int ci = i - cx, cj = j - cy, ck = k - cz;
                    if (ci < 0 || cj < 0 || ck < 0 || ci > g.nn.x - 2 || cj > g.nn.y - 2 || ck > g.nn.z - 2) continue;
                    const int va = cx + 2 * cy + 4 * cz;
                    for (int vb = 0; vb < 8; ++vb) {
                        const int nb = node_of(g, ci + (vb & 1), cj + ((vb >> 1) & 1), ck + (vb >> 2));
                        const double *kb = kcell + (va * 8 + vb) * 9;
                        const double v0 = operand(u, u2, beta, (size_t)nb * 3), v1 = operand(u, u2, beta, (size_t)nb * 3 + 1),
                                     v2 = operand(u, u2, beta, (size_t)nb * 3 + 2);
                        y[0] += kb[0] * v0 + kb[1] * v1 + kb[2] * v2;
                        y[1] += kb[3] * v0 + kb[4] * v1 + kb[5] * v2;
                        y[2] += kb[6] * v0 + kb[7] * v1 + kb[8] * v2;
                    }
                }
    }
    if (with_w) {
        const double *wr = wst + (size_t)node_of(g, i, j, k) * 27;
        for (int dk = -1; dk <= 1; ++dk)
            for (int dj = -1; dj <= 1; ++dj)
                for (int di = -1; di <= 1; ++di) {
                    const double wv = wr[(di + 1) + 3 * (dj + 1) + 9 * (dk + 1)];
                    if (wv == 0.0) continue;            // also skips neighbours outside the grid (never written)
                    const int nb = node_of(g, i + di, j + dj, k + dk);
                    y[0] += wv * operand(u, u2, beta, (size_t)nb * 3);
                    y[1] += wv * operand(u, u2, beta, (size_t)nb * 3 + 1);
                    y[2] += wv * operand(u, u2, beta, (size_t)nb * 3 + 2);
                }
    }
}

__device__ __forceinline__ void node_ijk(const FemGeom &g, int node, int &i, int &j, int &k)
{
    const int nxy = g.nn.x * g.nn.y;
    k = node / nxy;
    j = (node - k * nxy) / g.nn.x;
    i = node - k * nxy - j * g.nn.x;
}

// diag(A) = diag(K) + diag(W)
__global__ void __launch_bounds__(kFemThreads)
fem_diag_kernel(FemGeom g, const double *__restrict__ kcell, const double *__restrict__ wst, double *diag)
{
    const int node = blockIdx.x * kFemThreads + threadIdx.x;
    if (node >= g.n) return;
    int i, j, k;
    node_ijk(g, node, i, j, k);
    double d[3] = {0.0, 0.0, 0.0};
    for (int cz = 0; cz < 2; ++cz)
        for (int cy = 0; cy < 2; ++cy)
            for (int cx = 0; cx < 2; ++cx) {
                const int ci = i - cx, cj = j - cy, ck = k - cz;
                if (ci < 0 || cj < 0 || ck < 0 || ci > g.nn.x - 2 || cj > g.nn.y - 2 || ck > g.nn.z - 2) continue;
                const int va = cx + 2 * cy + 4 * cz;
                const double *kb = kcell + (va * 8 + va) * 9;
                d[0] += kb[0]; d[1] += kb[4]; d[2] += kb[8];
            }
    const double wv = wst[(size_t)node * 27 + 13];
    diag[(size_t)node * 3] = d[0] + wv;
    diag[(size_t)node * 3 + 1] = d[1] + wv;
    diag[(size_t)node * 3 + 2] = d[2] + wv;
}

// Sum over the CTA in a fixed order (kFemThreads = 4 warps); every thread gets the total.
__device__ double cta_sum(double v, double *s_red)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
    for (int w = 0; w < kFemThreads / 32; ++w) t += s_red[w];
    return t;
}

// Writes this CTA's partial sums; returns true in the last CTA to arrive, with `tot` = the sums over all CTAs in CTA
// order (a fixed order: the result does not depend on which CTA happens to be last).
template <int NV>
__device__ bool finish_sums(const double (&part)[NV], double *parts, PcgState *st, double (&tot)[NV])
{
    __shared__ bool s_last;
    if (threadIdx.x == 0) {
        for (int v = 0; v < NV; ++v) parts[(size_t)v * kMaxParts + blockIdx.x] = part[v];
        __threadfence();
        s_last = atomicAdd(&st->ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!s_last) return false;
    __threadfence();
    if (threadIdx.x == 0) {
        for (int v = 0; v < NV; ++v) {
            double t = 0.0;
            for (unsigned int c = 0; c < gridDim.x; ++c) t += __ldcg(parts + (size_t)v * kMaxParts + c);
            tot[v] = t;
        }
        st->ticket = 0u;
    }
    return true;
}

// b = rhs0 + K x (the force F_i of PAPER.md:258);  r = b - A x;  z = r / diag;  p = z;  rz, rr, bb
__global__ void __launch_bounds__(kFemThreads)
pcg_init_kernel(FemGeom g, const double *__restrict__ kcell, const double *__restrict__ wst, const double *__restrict__ rhs0,
                const double *__restrict__ diag, const double *__restrict__ x, double *b, double *r, double *z, double *p,
                double *parts, PcgState *st, double tol)
{
    __shared__ double s_red[kFemThreads / 32];
    const int node = blockIdx.x * kFemThreads + threadIdx.x;
    double rz = 0.0, rr = 0.0, bb = 0.0;
    if (node < g.n) {
        int i, j, k;
        node_ijk(g, node, i, j, k);
        double kx[3], wx[3];
        apply_node(g, kcell, wst, x, i, j, k, true, false, kx);
        apply_node(g, kcell, wst, x, i, j, k, false, true, wx);
        for (int a = 0; a < 3; ++a) {
            const size_t e = (size_t)node * 3 + a;
            const double bv = rhs0[e] + kx[a];
            const double rv = rhs0[e] - wx[a];            // b - (K + W) x
            const double dv = diag[e];
            const double zv = dv > 0.0 ? rv / dv : 0.0;
            b[e] = bv; r[e] = rv; z[e] = zv; p[e] = zv;
            rz += rv * zv; rr += rv * rv; bb += bv * bv;
        }
    }
    const double part[3] = {cta_sum(rz, s_red), cta_sum(rr, s_red), cta_sum(bb, s_red)};
    double tot[3];
    if (finish_sums<3>(part, parts, st, tot) && threadIdx.x == 0) {
        st->rz = tot[0]; st->rr = tot[1]; st->bb = tot[2];
        st->tol2 = tol * tol;
        st->beta = 0.0;                                   // the first direction is z itself
        st->iters = 0;
        st->done = tot[1] <= tol * tol * tot[2] ? 1 : 0;
    }
}

// p = z + beta p_old (written to the OTHER buffer: neighbours still read p_old);  q = A p;  pq = p . q;  alpha = rz / pq.
// The direction update is fused into the operator application: p at a neighbour is formed on the fly from z and p_old.
__global__ void __launch_bounds__(kFemThreads)
pcg_apply_kernel(FemGeom g, const double *__restrict__ kcell, const double *__restrict__ wst, const double *__restrict__ z,
                 const double *__restrict__ p_old, double *__restrict__ p_new, double *q, double *parts, PcgState *st)
{
    __shared__ double s_red[kFemThreads / 32];
    if (st->done) return;                                 // uniform over the grid: written by an earlier launch
    const double beta = st->beta;
    const int node = blockIdx.x * kFemThreads + threadIdx.x;
    double pq = 0.0;
    if (node < g.n) {
        int i, j, k;
        node_ijk(g, node, i, j, k);
        double y[3], yw[3];
        apply_node(g, kcell, wst, z, i, j, k, true, false, y, p_old, beta);
        apply_node(g, kcell, wst, z, i, j, k, false, true, yw, p_old, beta);
        for (int a = 0; a < 3; ++a) {
            const size_t e = (size_t)node * 3 + a;
            const double pv = operand(z, p_old, beta, e);
            const double qv = y[a] + yw[a];
            p_new[e] = pv;
            q[e] = qv;
            pq += pv * qv;
        }
    }
    const double part[1] = {cta_sum(pq, s_red)};
    double tot[1];
    if (finish_sums<1>(part, parts, st, tot) && threadIdx.x == 0) {
        st->pq = tot[0];
        st->alpha = tot[0] > 0.0 ? st->rz / tot[0] : 0.0;
    }
}

// x += alpha p;  r -= alpha q;  z = r / diag;  rz', rr;  beta = rz' / rz;  convergence
__global__ void __launch_bounds__(kFemThreads)
pcg_update_kernel(FemGeom g, const double *__restrict__ diag, const double *__restrict__ p, const double *__restrict__ q,
                  double *x, double *r, double *z, double *parts, PcgState *st)
{
    __shared__ double s_red[kFemThreads / 32];
    if (st->done) return;
    const double alpha = st->alpha;
    const int node = blockIdx.x * kFemThreads + threadIdx.x;
    double rz = 0.0, rr = 0.0;
    if (node < g.n)
        for (int a = 0; a < 3; ++a) {
            const size_t e = (size_t)node * 3 + a;
            x[e] += alpha * p[e];
            const double rv = r[e] - alpha * q[e];
            const double dv = diag[e];
            const double zv = dv > 0.0 ? rv / dv : 0.0;
            r[e] = rv; z[e] = zv;
            rz += rv * zv; rr += rv * rv;
        }
    const double part[2] = {cta_sum(rz, s_red), cta_sum(rr, s_red)};
    double tot[2];
    if (finish_sums<2>(part, parts, st, tot) && threadIdx.x == 0) {
        st->beta = st->rz > 0.0 ? tot[0] / st->rz : 0.0;
        st->rz = tot[0];
        st->rr = tot[1];
        st->iters += 1;
        if (tot[1] <= st->tol2 * st->bb) st->done = 1;
    }
}

// field[c][voxel] = sum_a w_a U[node_a][c]  (fp32: what nrr_bm_warp takes)
__global__ void __launch_bounds__(256)
fem_dense_field_kernel(FemGeom g, const double *__restrict__ u, float *__restrict__ field)
{
    const size_t nvox = (size_t)g.dims.x * g.dims.y * g.dims.z;
    const size_t v = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (v >= nvox) return;
    const int x = (int)(v % g.dims.x), y = (int)((v / g.dims.x) % g.dims.y), z = (int)(v / ((size_t)g.dims.x * g.dims.y));
    int node[4];
    double w[4];
    locate(g, (double)x, (double)y, (double)z, node, w);
    for (int c = 0; c < 3; ++c) {
        double s = 0.0;
        for (int a = 0; a < 4; ++a) s += w[a] * u[(size_t)node[a] * 3 + c];
        field[(size_t)c * nvox + v] = (float)s;
    }
}

}  // namespace

struct nrr_bm_fem {
    unsigned int magic = 0;
    int device = 0;
    FemGeom g{};
    double young = 0.0, poisson = 0.0;
    double *kcell = nullptr, *wst = nullptr, *rhs0 = nullptr, *diag = nullptr;
    double *x = nullptr, *b = nullptr, *r = nullptr, *z = nullptr, *p = nullptr, *p2 = nullptr, *q = nullptr, *parts = nullptr;
    PcgState *st = nullptr;
};

namespace {

constexpr unsigned int kFemMagic = 0x4e524646u;      // "NRFF"

void fem_free(nrr_bm_fem *f)
{
    if (!f) return;
    void *bufs[] = {f->kcell, f->wst, f->rhs0, f->diag, f->x, f->b, f->r, f->z, f->p, f->p2, f->q, f->parts, f->st};
    for (void *p : bufs)
        if (p) cudaFree(p);
    f->magic = 0;
    delete f;
}

int fem_ok(const nrr_bm_fem *f)
{
    if (!f || f->magic != kFemMagic) return api_fail(NRR_E_ARG, "not a live nrr_bm_fem");
    int dev = 0;
    NRR_CUDA(cudaGetDevice(&dev));
    if (dev != f->device) return api_fail(NRR_E_ARG, "the model belongs to device %d, the current device is %d", f->device, dev);
    return NRR_OK;
}

int fem_solve_device(nrr_bm_fem *f, const int *blocks, const int *disp, const float *ncc, int n, double weight, int n_iter,
                     double tol, int max_cg, double *out_u, int *out_cg_iters, cudaStream_t stream)
{
    void *pinned = nullptr;
    int rc = api_thread_state(nullptr, &pinned);
    if (rc) return rc;
    const FemGeom g = f->g;
    const int ctas = (g.n + kFemThreads - 1) / kFemThreads, n3 = 3 * g.n;
    NRR_CUDA(cudaMemsetAsync(f->wst, 0, sizeof(double) * 27 * (size_t)g.n, stream));
    NRR_CUDA(cudaMemsetAsync(f->rhs0, 0, sizeof(double) * (size_t)n3, stream));
    NRR_CUDA(cudaMemsetAsync(f->x, 0, sizeof(double) * (size_t)n3, stream));      // U_0 = 0
    NRR_CUDA(cudaMemsetAsync(f->st, 0, sizeof(PcgState), stream));
    if (n > 0) {
        NRR_LAUNCH(fem_accumulate_kernel, (n + kFemThreads - 1) / kFemThreads, kFemThreads, 0, stream, g, blocks, disp, ncc, n,
                   weight, f->wst, f->rhs0);
        NRR_LAUNCH_CHECK("fem_accumulate_kernel");
    }
    NRR_LAUNCH(fem_diag_kernel, ctas, kFemThreads, 0, stream, g, f->kcell, f->wst, f->diag);
    NRR_LAUNCH_CHECK("fem_diag_kernel");
    PcgState *h = (PcgState *)pinned;
    int total_iters = 0;
    bool converged = true;
    for (int outer = 0; outer < n_iter; ++outer) {
        // F_i = K U_i enters the right-hand side; the solve starts from U_i
        NRR_LAUNCH(pcg_init_kernel, ctas, kFemThreads, 0, stream, g, f->kcell, f->wst, f->rhs0, f->diag, f->x, f->b, f->r, f->z,
                   f->p, f->parts, f->st, tol);
        NRR_LAUNCH_CHECK("pcg_init_kernel");
        int it = 0, cur = 0;                               // pcg_init_kernel wrote the first direction into pbuf[0]
        double *pbuf[2] = {f->p, f->p2};
        bool done = false;
        while (!done && it < max_cg) {
            const int batch = max_cg - it < 16 ? max_cg - it : 16;      // one host poll per 16 iterations
            for (int s = 0; s < batch; ++s) {      // two launches per iteration; the direction ping-pongs between two buffers
                double *p_old = pbuf[cur], *p_new = pbuf[cur ^ 1];
                NRR_LAUNCH(pcg_apply_kernel, ctas, kFemThreads, 0, stream, g, f->kcell, f->wst, f->z, p_old, p_new, f->q, f->parts, f->st);
                NRR_LAUNCH_CHECK("pcg_apply_kernel");
                NRR_LAUNCH(pcg_update_kernel, ctas, kFemThreads, 0, stream, g, f->diag, p_new, f->q, f->x, f->r, f->z, f->parts, f->st);
                NRR_LAUNCH_CHECK("pcg_update_kernel");
                cur ^= 1;
            }
            it += batch;
            NRR_CUDA(cudaMemcpyAsync(h, f->st, sizeof(PcgState), cudaMemcpyDeviceToHost, stream));
            NRR_CUDA(cudaStreamSynchronize(stream));
            done = h->done != 0;
        }
        total_iters += h->iters;
        if (!done) converged = false;
    }
    if (out_u) NRR_CUDA(cudaMemcpyAsync(out_u, f->x, sizeof(double) * (size_t)n3, cudaMemcpyDeviceToDevice, stream));
    if (out_cg_iters) *out_cg_iters = total_iters;
    if (!converged) return api_fail(NRR_E_NOCONV, "conjugate gradients did not reach tol = %g within %d iterations (|r|^2 = %g, |b|^2 = %g)",
                                    tol, max_cg, h->rr, h->bb);
    return NRR_OK;
}

int check_solve_args(const nrr_bm_fem *f, const int *blocks, const int *disp, const float *ncc, int n, double weight, int n_iter,
                     double tol, int max_cg)
{
    if (!f || f->magic != kFemMagic) return api_fail(NRR_E_ARG, "not a live nrr_bm_fem");
    if (n < 0) return api_fail(NRR_E_ARG, "n = %d < 0", n);
    if (n > 0 && (!blocks || !disp || !ncc)) return api_fail(NRR_E_NULL, "blocks/disp/ncc is NULL with n > 0");
    if (!(weight >= 0.0)) return api_fail(NRR_E_ARG, "weight = %g < 0", weight);
    if (n_iter < 1) return api_fail(NRR_E_ARG, "n_iter = %d < 1", n_iter);
    if (!(tol > 0.0 && tol < 1.0)) return api_fail(NRR_E_ARG, "tol = %g outside (0, 1)", tol);
    if (max_cg < 1) return api_fail(NRR_E_ARG, "max_cg = %d < 1", max_cg);
    return NRR_OK;
}

}  // namespace

extern "C" {

int nrr_bm_fem_create(const int dims[3], const int spacing[3], double young, double poisson, nrr_bm_fem **out_fem)
{
    if (!out_fem) return api_fail(NRR_E_NULL, "out_fem is NULL");
    *out_fem = nullptr;
    if (!dims || !spacing) return api_fail(NRR_E_NULL, "dims/spacing is NULL");
    for (int a = 0; a < 3; ++a) {
        if (dims[a] < 1) return api_fail(NRR_E_DIMS, "dims[%d] = %d < 1", a, dims[a]);
        if (spacing[a] < 1) return api_fail(NRR_E_STRIDE, "spacing[%d] = %d < 1", a, spacing[a]);
    }
    if (!(young >= 0.0)) return api_fail(NRR_E_ARG, "young = %g < 0", young);
    if (!(poisson > -1.0 && poisson < 0.5)) return api_fail(NRR_E_ARG, "poisson = %g outside (-1, 0.5)", poisson);
    FemGeom g;
    g.dims = Int3{dims[0], dims[1], dims[2]};
    g.h = Int3{spacing[0], spacing[1], spacing[2]};
    int nn[3];
    for (int a = 0; a < 3; ++a) {
        nn[a] = (dims[a] - 1 + spacing[a] - 1) / spacing[a] + 1;
        if (nn[a] < 2) nn[a] = 2;
    }
    g.nn = Int3{nn[0], nn[1], nn[2]};
    const long long n = (long long)nn[0] * nn[1] * nn[2];
    if (n > (long long)kMaxParts * kFemThreads) return api_fail(NRR_E_DIMS, "the mesh has %lld nodes (limit %d)", n, kMaxParts * kFemThreads);
    g.n = (int)n;
    nrr_bm_fem *f = new nrr_bm_fem();
    f->magic = kFemMagic;
    f->g = g;
    f->young = young; f->poisson = poisson;
    auto fail_with = [&](int code) { fem_free(f); return code; };
    if (cudaGetDevice(&f->device) != cudaSuccess) return fail_with(api_fail(NRR_E_CUDA, "no CUDA device"));
    const size_t n3 = 3 * (size_t)g.n;
    double **vecs[] = {&f->rhs0, &f->diag, &f->x, &f->b, &f->r, &f->z, &f->p, &f->p2, &f->q};
    bool ok = cudaMalloc((void **)&f->kcell, sizeof(double) * 8 * 8 * 9) == cudaSuccess &&
              cudaMalloc((void **)&f->wst, sizeof(double) * 27 * (size_t)g.n) == cudaSuccess &&
              cudaMalloc((void **)&f->parts, sizeof(double) * 3 * kMaxParts) == cudaSuccess &&
              cudaMalloc((void **)&f->st, sizeof(PcgState)) == cudaSuccess;
    for (double **v : vecs) ok = ok && cudaMalloc((void **)v, sizeof(double) * n3) == cudaSuccess;
    if (!ok) return fail_with(api_fail(NRR_E_CUDA, "cudaMalloc of the model's vectors failed"));
    const double lam = young * poisson / ((1.0 + poisson) * (1.0 - 2.0 * poisson)), mu = young / (2.0 * (1.0 + poisson));
    NRR_LAUNCH(fem_cell_kernel, 1, 64, 0, (cudaStream_t) nullptr, (double)spacing[0], (double)spacing[1], (double)spacing[2], lam, mu, f->kcell);
    if (cudaGetLastError() != cudaSuccess || cudaDeviceSynchronize() != cudaSuccess) return fail_with(api_fail(NRR_E_CUDA, "fem_cell_kernel failed"));
    count_launch();
    *out_fem = f;
    return NRR_OK;
}

int nrr_bm_fem_info(const nrr_bm_fem *fem, int nodes[3], int *n_nodes)
{
    if (!fem || fem->magic != kFemMagic) return api_fail(NRR_E_ARG, "not a live nrr_bm_fem");
    if (nodes) { nodes[0] = fem->g.nn.x; nodes[1] = fem->g.nn.y; nodes[2] = fem->g.nn.z; }
    if (n_nodes) *n_nodes = fem->g.n;
    return NRR_OK;
}

int nrr_bm_fem_solve(nrr_bm_fem *fem, const int *blocks, const int *disp, const float *ncc, int n, double weight, int n_iter,
                     double tol, int max_cg, double *out_u, int *out_cg_iters, void *stream)
{
    int rc = check_solve_args(fem, blocks, disp, ncc, n, weight, n_iter, tol, max_cg);
    if (rc) return rc;
    if (!out_u) return api_fail(NRR_E_NULL, "out_u is NULL");
    if ((rc = fem_ok(fem))) return rc;
    return fem_solve_device(fem, blocks, disp, ncc, n, weight, n_iter, tol, max_cg, out_u, out_cg_iters, (cudaStream_t)stream);
}

int nrr_bm_fem_solve_host(nrr_bm_fem *fem, const int *blocks, const int *disp, const float *ncc, int n, double weight,
                          int n_iter, double tol, int max_cg, double *out_u, int *out_cg_iters)
{
    int rc = check_solve_args(fem, blocks, disp, ncc, n, weight, n_iter, tol, max_cg);
    if (rc) return rc;
    if (!out_u) return api_fail(NRR_E_NULL, "out_u is NULL");
    if ((rc = fem_ok(fem))) return rc;
    cudaStream_t s;
    if ((rc = api_host_stream(&s))) return rc;
    AsyncScratch d_blocks(s), d_disp(s), d_ncc(s);
    const size_t n1 = (size_t)(n > 0 ? n : 1);
    NRR_CUDA(d_blocks.alloc(n1 * 3 * sizeof(int)));
    NRR_CUDA(d_disp.alloc(n1 * 3 * sizeof(int)));
    NRR_CUDA(d_ncc.alloc(n1 * sizeof(float)));
    if (n > 0) {
        NRR_CUDA(cudaMemcpyAsync(d_blocks.p, blocks, (size_t)n * 3 * sizeof(int), cudaMemcpyHostToDevice, s));
        NRR_CUDA(cudaMemcpyAsync(d_disp.p, disp, (size_t)n * 3 * sizeof(int), cudaMemcpyHostToDevice, s));
        NRR_CUDA(cudaMemcpyAsync(d_ncc.p, ncc, (size_t)n * sizeof(float), cudaMemcpyHostToDevice, s));
    }
    rc = fem_solve_device(fem, (const int *)d_blocks.p, (const int *)d_disp.p, (const float *)d_ncc.p, n, weight, n_iter, tol,
                          max_cg, nullptr, out_cg_iters, s);
    if (rc != NRR_OK && rc != NRR_E_NOCONV) return rc;
    NRR_CUDA(cudaMemcpyAsync(out_u, fem->x, sizeof(double) * 3 * (size_t)fem->g.n, cudaMemcpyDeviceToHost, s));
    NRR_CUDA(cudaStreamSynchronize(s));
    return rc;
}

int nrr_bm_fem_dense_field(const nrr_bm_fem *fem, const double *u, float *out_field, void *stream)
{
    int rc = fem_ok(fem);
    if (rc) return rc;
    if (!u || !out_field) return api_fail(NRR_E_NULL, "u/out_field is NULL");
    const size_t nvox = (size_t)fem->g.dims.x * fem->g.dims.y * fem->g.dims.z;
    const FemGeom g = fem->g;
    NRR_LAUNCH(fem_dense_field_kernel, (unsigned int)((nvox + 255) / 256), 256, 0, (cudaStream_t)stream, g, u, out_field);
    NRR_LAUNCH_CHECK("fem_dense_field_kernel");
    return NRR_OK;
}

int nrr_bm_fem_dense_field_host(const nrr_bm_fem *fem, const double *u, float *out_field)
{
    int rc = fem_ok(fem);
    if (rc) return rc;
    if (!u || !out_field) return api_fail(NRR_E_NULL, "u/out_field is NULL");
    cudaStream_t s;
    if ((rc = api_host_stream(&s))) return rc;
    const size_t nvox = (size_t)fem->g.dims.x * fem->g.dims.y * fem->g.dims.z, n3 = 3 * (size_t)fem->g.n;
    AsyncScratch d_u(s), d_f(s);
    NRR_CUDA(d_u.alloc(n3 * sizeof(double)));
    NRR_CUDA(d_f.alloc(3 * nvox * sizeof(float)));
    NRR_CUDA(cudaMemcpyAsync(d_u.p, u, n3 * sizeof(double), cudaMemcpyHostToDevice, s));
    const double *du = (const double *)d_u.p;
    float *df = (float *)d_f.p;
    const FemGeom g = fem->g;
    NRR_LAUNCH(fem_dense_field_kernel, (unsigned int)((nvox + 255) / 256), 256, 0, s, g, du, df);
    NRR_LAUNCH_CHECK("fem_dense_field_kernel");
    NRR_CUDA(cudaMemcpyAsync(out_field, d_f.p, 3 * nvox * sizeof(float), cudaMemcpyDeviceToHost, s));
    NRR_CUDA(cudaStreamSynchronize(s));
    return NRR_OK;
}

int nrr_bm_fem_destroy(nrr_bm_fem *fem)
{
    if (!fem) return NRR_OK;
    if (fem->magic != kFemMagic) return api_fail(NRR_E_ARG, "not a live nrr_bm_fem");
    cudaDeviceSynchronize();
    fem_free(fem);
    return NRR_OK;
}

}  // extern "C"
