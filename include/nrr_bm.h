/*
 * nrr_bm.h -- C ABI of the B200-native block-matching library (libnrr_bm.so).
 *
 * The data-parallel hot path of the physics-based non-rigid registration of arxiv/paper_2308_10868:
 * variance-based block ("feature") selection in the pre-operative image and exhaustive NCC block matching
 * against the intra-operative image.  Everything below runs in hand-written CUDA kernels for sm_100a; there
 * is no CPU fallback: without a CUDA device every compute entry point returns NRR_E_CUDA.
 *
 * NAMES (BASELINE.json / SURVEY.md section 0).  The paper and this ABI use opposite image names:
 *   "fixed"  = the paper's FLOATING / pre-operative image: blocks are selected and cut here
 *              (section 3);
 *   "moving" = the paper's REFERENCE / target / intra-operative image: the search window lives here
 *              (listing PAPER.md:660-662, section 4.3 "search window sw in fixed image").
 *
 * LAYOUT.  A volume with dims = (nx, ny, nz) is a dense fp32 array, voxel (x,y,z) at (z*ny + y)*nx + x
 * (x fastest).  Both volumes share dims (rigidly pre-aligned images on a common grid).
 * All triples (dims, block, stride, window, block centres, displacements) are in (x, y, z) order.
 *
 * POINTERS.  In the device entry points every volume / array pointer is a DEVICE pointer owned by the
 * caller (e.g. a torch tensor); dims/block/stride/window and out_n are HOST pointers.  In the *_host entry
 * points every pointer is a HOST pointer.  `stream` is a cudaStream_t passed as void* (NULL = the legacy
 * default stream).  The library never frees or retains caller pointers past the stream-ordered completion
 * of the call; internal scratch is library-owned, allocated stream-ordered (cudaMallocAsync) and reused.
 *
 * ERRORS.  Every entry point returns NRR_OK (0) or a negative nrr_status; no exception crosses the ABI.
 * nrr_bm_last_error() returns a thread-local message for the last nonzero return on this thread.
 */
#ifndef NRR_BM_H
#define NRR_BM_H

#ifdef __cplusplus
extern "C" {
#endif

#define NRR_BM_VERSION 200 /* 0.2.0 : major*10000 + minor*100 + patch */

#if defined(__GNUC__)
#define NRR_BM_API __attribute__((visibility("default")))
#else
#define NRR_BM_API
#endif

typedef enum nrr_status {
    NRR_OK = 0,
    NRR_E_NULL = -1,     /* a required pointer is NULL */
    NRR_E_DIMS = -2,     /* a dimension is < 1, or the block is larger than the volume */
    NRR_E_BLOCK = -3,    /* a block edge is < 1 or even (centres need odd edges; the paper parameterises
                            blocks by a half size) */
    NRR_E_STRIDE = -4,   /* a stride is < 1 */
    NRR_E_WINDOW = -5,   /* a window half-range is < 0 */
    NRR_E_FRAC = -6,     /* frac outside (0, 1] */
    NRR_E_CAPACITY = -7, /* K > capacity; *out_n is still set to K, out_blocks holds the first `capacity` */
    NRR_E_BOUNDS = -8,   /* a supplied block leaves the volume (validated on the device; reported by the
                            synchronising host entry points and by nrr_bm_check_async_error) */
    NRR_E_SMEM = -9,     /* block / window too large for the kernels' shared-memory or index limits */
    NRR_E_CUDA = -10,    /* a CUDA runtime call failed (message in nrr_bm_last_error) */
    NRR_E_ARG = -11,     /* other invalid argument (n < 0, capacity < 0, ...) */
    NRR_E_NOCONV = -13,  /* nrr_bm_fem_solve: conjugate gradients did not reach the tolerance within max_cg iterations
                            (out_u holds the last iterate) */
    NRR_E_DEVICE = -12   /* a staged copy of a matching kernel did not complete within its time bound; the blocks
                            of that CTA get out_disp = (0,0,0), out_ncc = NaN.  Reported like NRR_E_BOUNDS (sticky
                            device flag); the kernel leaves in an orderly way and never faults the GPU */
} nrr_status;

/*
 * Variance-based block selection  --  PAPER.md:231-236 (section 3: registration points are where "the
 * variability in the intensities in the surrounding region exceeds some threshold", identified "prior to
 * the time-critical part") and PAPER.md:376 (section 4.1: "computes the variance within a block of size
 * B_s", "selects F_s features with the highest variance", "0.5 + NFeatures x Fs blocks are selected").
 *
 * Candidates: the stride grid from origin 0 with blocks fully inside the volume, in ascending linear grid
 * order (x fastest); a grid position is a candidate iff mask == NULL or mask[centre voxel] != 0; the
 * population variance is taken over the whole block regardless of the mask.  With N candidates,
 * K = floor(0.5 + N*frac) are kept: those of largest variance, ties to the lower candidate index.
 *
 *   fixed      [in]  device fp32 [nz][ny][nx]
 *   dims       [in]  host int[3] (nx, ny, nz)
 *   block      [in]  host int[3] full odd edge length per axis
 *   stride     [in]  host int[3] grid stride per axis, >= 1
 *   frac       [in]  selection fraction F_s in (0, 1]
 *   mask       [in]  device uint8 [nz][ny][nx], or NULL (= every voxel)
 *   out_blocks [out] device int32 [capacity][3]: block CENTRES (origin + (B-1)/2) of the kept candidates in
 *                    ascending candidate index (a set with a canonical listing)
 *   capacity   [in]  rows available in out_blocks / out_var
 *   out_n      [out] HOST int: K.  The call synchronises `stream` once to return it.
 *   out_var    [out] device double [capacity], or NULL: population variance of each kept block, same order
 *   out_ncand  [out] HOST int, or NULL: N, the number of candidates
 */
NRR_BM_API int nrr_bm_select_blocks(const float *fixed, const int dims[3], const int block[3], const int stride[3],
                         double frac, const unsigned char *mask, int *out_blocks, int capacity, int *out_n,
                         double *out_var, int *out_ncand, void *stream);

/*
 * Selection under the paper's connectivity pattern  --  PAPER.md:376 (section 4.1): "The method also uses a
 * connectivity pattern to avoid selecting blocks that are too close to each other ... vertex (26 connectivity),
 * edge (18 connectivity), face (6 connectivity)".  The paper names the patterns, not the algorithm; this library
 * reads it (Q20) as the greedy walk by (variance descending, candidate index ascending) that keeps a
 * candidate iff none of its pattern neighbours ON THE CANDIDATE GRID (grid offsets with |di|+|dj|+|dk| <= 1 / 2
 * / 3 for 6 / 18 / 26) is kept already, and stops at K = floor(0.5 + N*frac) kept or at the end of the list.
 * With stride 1 (the paper's setting: every intracranial voxel is a candidate) the grid neighbours are the voxel
 * neighbours of the block centre.  connectivity = 0 is nrr_bm_select_blocks.  Everything else (candidates,
 * variance, outputs in ascending candidate index, *out_n on the HOST) as in nrr_bm_select_blocks; *out_n can be
 * below K when the pattern leaves fewer candidates.  The call synchronises `stream` several times (it polls
 * the device between batches of pruning rounds); selection is pre-operative.
 */
NRR_BM_API int nrr_bm_select_blocks_pruned(const float *fixed, const int dims[3], const int block[3],
                                const int stride[3], double frac, const unsigned char *mask, int connectivity,
                                int *out_blocks, int capacity, int *out_n, double *out_var, int *out_ncand,
                                void *stream);
NRR_BM_API int nrr_bm_select_blocks_pruned_host(const float *fixed, const int dims[3], const int block[3],
                                     const int stride[3], double frac, const unsigned char *mask, int connectivity,
                                     int *out_blocks, int capacity, int *out_n, double *out_var, int *out_ncand);

/*
 * Exhaustive NCC block matching  --  PAPER.md:236-246 (section 3: for each registration point, the block
 * displacement "that maximizes the intensity-based similarity metric", NCC equation) and the listing
 * PAPER.md:659-667 (section 4.3: for each block, each candidate block in the window, similarity, maximum
 * and its displacement).  Cost bound O(BxByBz x WxWyWz) per point.
 *
 * For block b with centre c and origin o = c - (B-1)/2, every displacement d with |d_a| <= window[a] whose
 * block at o+d stays inside the moving volume is evaluated (others are skipped);
 *     NCC(d) = sum (f - fbar)(m - mbar) / sqrt( sum (f - fbar)^2 * sum (m - mbar)^2 )
 * over the B voxels of the fixed block at o and the moving block at o+d; a zero-variance block scores 0.
 * out_disp[b] = the d of largest NCC (equal maxima: lowest linear candidate index
 * ((dz+rz)(2ry+1) + (dy+ry))(2rx+1) + (dx+rx)), out_ncc[b] = that NCC.  fixed(p+v) ~ moving(p+d+v);
 * units are voxels.  out_ncc is the confidence S of PAPER.md:263-264 in raw form.
 *
 *   fixed, moving [in]  device fp32 [nz][ny][nx]
 *   blocks        [in]  device int32 [n][3] block centres (as written by nrr_bm_select_blocks)
 *   n             [in]  number of blocks, >= 0
 *   block         [in]  host int[3] full odd edge length per axis
 *   window        [in]  host int[3] displacement half-range r per axis, >= 0; candidates = prod(2r+1)
 *   out_disp      [out] device int32 [n][3]
 *   out_ncc       [out] device fp32 [n]
 * Asynchronous: kernels are enqueued on `stream` and the call returns.  A block that leaves the volume gets
 * out_disp = (0,0,0), out_ncc = NaN and raises a sticky device flag that nrr_bm_check_async_error reports.
 */
NRR_BM_API int nrr_bm_match(const float *fixed, const float *moving, const int dims[3], const int *blocks, int n,
                 const int block[3], const int window[3], int *out_disp, float *out_ncc, void *stream);

/*
 * Selection + matching of one volume pair in ONE asynchronous call (no host synchronisation at all): the
 * selection kernels, the moving-volume statistics and the matching kernels are enqueued back to back; the
 * matching kernels are launched for the host-side upper bound floor(0.5 + grid positions * frac) on K and read
 * K itself from device memory.  This is the call for pipelines and parameter sweeps that must not stall the
 * stream (BASELINE.json config 5: 32 settings "in one launch sequence").  Arguments as in nrr_bm_select_blocks
 * and nrr_bm_match, except
 *   out_n  [out] DEVICE int (nullable): K.  If K > capacity only the first `capacity` blocks (ascending
 *                candidate index) are written and matched; the caller sees K > capacity after its own sync.
 * Rows [K, capacity) of out_blocks / out_disp / out_ncc are left untouched.
 */
NRR_BM_API int nrr_bm_register(const float *fixed, const float *moving, const int dims[3], const int block[3],
                    const int stride[3], const int window[3], double frac, const unsigned char *mask, int *out_blocks,
                    int capacity, int *out_n, int *out_disp, float *out_ncc, void *stream);

/*
 * Per-candidate normalisers of the moving volume (row M2 of the hot path; nrr_bm_match runs this itself,
 * the entry point exposes it for tests and for callers that match one moving volume against many block lists).
 * For every block ORIGIN p whose block fits in the volume,
 *     out_inv_sd[p] = 1 / sqrt( sum over the block at p of (m - mean)^2 ),   0 for a zero-variance block,
 * i.e. the moving-image factor of NCC's denominator; entries whose block would leave the
 * volume are left untouched.  Sums are accumulated in FP64; the result is rounded to fp32.
 *   moving      [in]  device fp32 [nz][ny][nx]        out_inv_sd [out] device fp32 [nz][ny][nx]
 * Asynchronous on `stream`.  nrr_bm_moving_stats_host: same with HOST buffers, synchronises.
 */
NRR_BM_API int nrr_bm_moving_stats(const float *moving, const int dims[3], const int block[3], float *out_inv_sd,
                        void *stream);
NRR_BM_API int nrr_bm_moving_stats_host(const float *moving, const int dims[3], const int block[3], float *out_inv_sd);

/*
 * Warp of an image by a dense displacement field  --  PAPER.md:225-229 (section 3: the registration derives a
 * "dense deformation field that defines transformation for each point in the image space") and PAPER.md:286
 * (APBNRR re-registers the warped image in every iteration).  The paper gives no formula; this library reads it
 * (Q21) as the backward warp on the output grid with trilinear interpolation and edge clamping:
 *     out(p) = T[image](p + v(p)),   v(p) = (field[0][p], field[1][p], field[2][p]) in voxels, (x, y, z) order,
 * the sample position clamped to [0, n_a - 1] per axis, T linear along x, then y, then z.
 *   image [in]  device fp32 [nz][ny][nx]          field [in] device fp32 [3][nz][ny][nx] (component-major)
 *   out   [out] device fp32 [nz][ny][nx], must not alias image
 * Asynchronous on `stream`.  fp32 arithmetic: |out - exact| <= 8 * 2^-24 * max|image|.  nrr_bm_warp_host: HOST
 * buffers, synchronises.
 */
NRR_BM_API int nrr_bm_warp(const float *image, const int dims[3], const float *field, float *out, void *stream);
NRR_BM_API int nrr_bm_warp_host(const float *image, const int dims[3], const float *field, float *out);

/*
 * Upper bound on K, for sizing out_blocks / out_disp / out_ncc before a call that does not return K on the host
 * (nrr_bm_register, nrr_bm_register_batch).  *out_grid = stride-grid positions (an upper bound on N),
 * *out_bound >= floor(0.5 + N*frac) for every N <= *out_grid  (count rule of PAPER.md:376).  Pure host arithmetic;
 * the method's formula lives in the library, not in its callers.  Either output may be NULL.
 */
NRR_BM_API int nrr_bm_capacity_bound(const int dims[3], const int block[3], const int stride[3], double frac,
                                     int *out_grid, int *out_bound);

/*
 * PLANS: the boundary split along the paper's timeline  --  PAPER.md:231-236 (section 3): registration points "can be
 * identified prior to the time-critical part of the computation in the floating (pre-operative) image.  Once the
 * reference (intra-operative) scan is available, the deformation vector is estimated at each of the selected
 * points by means of block matching", and PAPER.md:267-268 ("block matching ... time critical and should be
 * performed while the surgeons are waiting").
 *
 *   nrr_bm_plan_create        PRE-OPERATIVE.  Everything that needs only the pre-operative (`fixed`) image: block
 *                             selection (S1-S3; connectivity = 0, 6, 18 or 26 as in nrr_bm_select_blocks_pruned), the
 *                             fixed-block records of the matching kernel (centred blocks, 1/sqrt(SS_f)), the kernel's
 *                             launch tables and all scratch.  Synchronises `stream`.
 *   nrr_bm_plan_match         INTRA-OPERATIVE, asynchronous on `stream`: the moving-volume normalisers (M2) and the
 *                             matching kernel (M1, M3-M5) for one intra-operative volume.  out_disp [n][3], out_ncc [n]
 *                             in the order of nrr_bm_plan_blocks.  Results are bit-identical to
 *                             nrr_bm_select_blocks + nrr_bm_match with the same arguments.
 *   nrr_bm_plan_match_range   the same for blocks [first, first + count) only; rows outside the range are left
 *                             untouched.  This is the natural shard of the path over several GPUs (PAPER.md:379-385:
 *                             both images on every processor, the block list distributed): rank r
 *                             holds a plan of its own, matches its slice and the ranks exchange 16 bytes per block.
 *   nrr_bm_plan_match_host    the same as nrr_bm_plan_match with HOST buffers (pinned memory makes the copies
 *                             asynchronous); synchronises.  The volume goes up in z slabs on a copy stream while the
 *                             normalisers and the matching of the blocks whose windows have landed already run, so
 *                             the call costs about one upload of `moving` plus the work on the last slab.
 *   nrr_bm_plan_destroy       releases everything the plan owns (NULL is allowed).
 *
 * OWNERSHIP.  nrr_bm_plan_create keeps the caller's `fixed` DEVICE pointer (the FP64 near-tie re-score reads the raw
 * voxels): it must stay valid and unchanged until nrr_bm_plan_destroy.  nrr_bm_plan_create_host takes HOST `fixed` /
 * `mask`, uploads them and owns the device copies.  A plan belongs to the device that was current at creation and
 * serves ONE match call at a time (calls on one stream are ordered by the stream; concurrent calls on several
 * streams must be ordered by the caller: they share the plan's scratch).  Errors as everywhere in this ABI;
 * NRR_E_ARG for a NULL / destroyed plan or a range outside [0, n].
 */
typedef struct nrr_bm_plan nrr_bm_plan;
NRR_BM_API int nrr_bm_plan_create(const float *fixed, const int dims[3], const int block[3], const int stride[3],
                                  const int window[3], double frac, const unsigned char *mask, int connectivity,
                                  void *stream, nrr_bm_plan **out_plan);
NRR_BM_API int nrr_bm_plan_create_host(const float *fixed, const int dims[3], const int block[3], const int stride[3],
                                       const int window[3], double frac, const unsigned char *mask, int connectivity,
                                       nrr_bm_plan **out_plan);
/* *out_n = K selected blocks, *out_ncand = N candidates (either may be NULL). */
NRR_BM_API int nrr_bm_plan_info(const nrr_bm_plan *plan, int *out_n, int *out_ncand);
/* Block centres [n][3] (ascending candidate index) and, if out_var != NULL, their variances [n]: HOST buffers. */
NRR_BM_API int nrr_bm_plan_blocks_host(const nrr_bm_plan *plan, int *out_blocks, double *out_var);
/* DEVICE pointer to the plan's block centres [n][3] (owned by the plan, valid until nrr_bm_plan_destroy). */
NRR_BM_API const int *nrr_bm_plan_blocks_device(const nrr_bm_plan *plan);
/* Copies the block centres [n][3] (and, if out_var != NULL, the variances [n]) into caller-owned DEVICE buffers,
 * asynchronously on `stream`. */
NRR_BM_API int nrr_bm_plan_blocks(const nrr_bm_plan *plan, int *out_blocks, double *out_var, void *stream);
NRR_BM_API int nrr_bm_plan_match(nrr_bm_plan *plan, const float *moving, int *out_disp, float *out_ncc, void *stream);
NRR_BM_API int nrr_bm_plan_match_range(nrr_bm_plan *plan, const float *moving, int first, int count, int *out_disp,
                                       float *out_ncc, void *stream);
NRR_BM_API int nrr_bm_plan_match_host(nrr_bm_plan *plan, const float *moving, int *out_disp, float *out_ncc);
NRR_BM_API int nrr_bm_plan_destroy(nrr_bm_plan *plan);

/*
 * PARAMETER SWEEP: one volume pair under many settings in ONE launch sequence  --  PAPER.md:527-540 (section 4.2,
 * speculative execution: "multiple instances of NRR are executed" with different parameter values) and PAPER.md:711
 * (block and window sizes are per-axis parameters); BASELINE.json configs[4].  No host synchronisation.  What the
 * settings have in common is computed once: the moving-volume normalisers per distinct block shape, the block
 * variances per distinct (block, stride) -- several fractions are selected from the same keys --, the fixed-block
 * records per distinct (block, stride, frac); the matching launches are spread over a few streams that fork from and
 * join into `stream`.  Per setting s the results are bit-identical to nrr_bm_register with that setting:
 *   out_blocks[s] [capacity[s]][3], out_disp[s] [capacity[s]][3], out_ncc[s] [capacity[s]]  DEVICE arrays (the arrays
 *   of pointers themselves are HOST arrays), out_n DEVICE int [n_settings]: K per setting.
 * Size capacity[s] with nrr_bm_capacity_bound.
 */
typedef struct nrr_bm_setting {
    int block[3];
    int stride[3];
    int window[3];
    double frac;
} nrr_bm_setting;
NRR_BM_API int nrr_bm_register_batch(const float *fixed, const float *moving, const int dims[3],
                                     const unsigned char *mask, const nrr_bm_setting *settings, int n_settings,
                                     int *const *out_blocks, const int *capacity, int *out_n, int *const *out_disp,
                                     float *const *out_ncc, void *stream);

/*
 * BIOMECHANICAL REGULARISATION of the sparse displacement field (the step that consumes out_disp / out_ncc)  --
 * PAPER.md:252-265 (section 3): "Estimation of brain deformation is based on the finite element analysis (FEA) using a
 * linear elastic model ... We then iteratively seek such a position of the mesh vertices U that balances the mechanical
 * forces of the modeled tissue that resist deformation, with the external forces that correspond to the displacements D
 * estimated by block matching:
 *        F_i <= K U_i ,      U_{i+1} <= [K + H^T S H]^-1 [H^T S D + F_i]
 * K is the mechanical stiffness matrix, H is the interpolation matrix from the mesh vertices to the block matching
 * displacements, S is the matrix that captures the confidence in the block matching results"; "Both
 * block matching and iterative estimation of displacements are time critical".
 *
 * Readings (Q22-Q25; the paper gives none of these).  MESH: the paper's mesher is out of scope; the model is a
 * regular grid of nodes, `spacing` voxels apart, covering the volume (nodes per axis = max(2, ceil((n-1)/spacing) + 1),
 * node index (k*nny + j)*nnx + i at position (i*hx, j*hy, k*hz) voxels), every cell cut into the six Kuhn tetrahedra
 * around its main diagonal, constant-strain elements.  MATERIAL: isotropic, Young's modulus `young` >= 0 and Poisson's
 * ratio `poisson` in (-1, 0.5) are inputs (the paper prints no constants).  S = weight * diag(max(NCC, 0)), one value per
 * block for its three axes; blocks with NCC <= 0 or NaN have no influence.  Displacements, positions and U in voxels.
 *
 *   nrr_bm_fem_create       builds the model (mesh geometry, the element stiffness table, all vectors) on the current device
 *   nrr_bm_fem_solve        U_0 = 0, then n_iter >= 1 iterations of the scheme above; each linear system is solved by
 *                           Jacobi-preconditioned conjugate gradients in FP64 to |r| <= tol * |b|, at most max_cg
 *                           iterations per system (NRR_E_NOCONV otherwise, with the last iterate in out_u).
 *                           blocks / disp int32 [n][3], ncc fp32 [n] as written by nrr_bm_select_blocks / nrr_bm_match
 *                           (DEVICE); out_u DEVICE double [n_nodes][3]; *out_cg_iters (HOST, nullable) = CG iterations
 *                           over all systems.  Synchronises `stream` (it polls the convergence flag every 16
 *                           iterations).  FP64 atomics accumulate H^T S H and H^T S D: bits can differ between runs in
 *                           the last places; against the oracle's direct solve |U - U_oracle| <= 1e-6 * max(1, max|U|)
 *                           for tol <= 1e-10.
 *   nrr_bm_fem_dense_field  "dense deformation field that defines transformation for each point in the image space"
 *                           (PAPER.md:225-229): out_field fp32 [3][nz][ny][nx] (component-major, what nrr_bm_warp
 *                           takes) = U interpolated at every voxel by the barycentric weights of its tetrahedron.
 *                           Asynchronous on `stream`.
 *   *_host                  the same with HOST buffers; synchronise.
 *   nrr_bm_fem_destroy      releases the model (NULL is allowed).
 */
typedef struct nrr_bm_fem nrr_bm_fem;
NRR_BM_API int nrr_bm_fem_create(const int dims[3], const int spacing[3], double young, double poisson, nrr_bm_fem **out_fem);
NRR_BM_API int nrr_bm_fem_info(const nrr_bm_fem *fem, int nodes[3], int *n_nodes);
NRR_BM_API int nrr_bm_fem_solve(nrr_bm_fem *fem, const int *blocks, const int *disp, const float *ncc, int n, double weight,
                                int n_iter, double tol, int max_cg, double *out_u, int *out_cg_iters, void *stream);
NRR_BM_API int nrr_bm_fem_solve_host(nrr_bm_fem *fem, const int *blocks, const int *disp, const float *ncc, int n,
                                     double weight, int n_iter, double tol, int max_cg, double *out_u, int *out_cg_iters);
NRR_BM_API int nrr_bm_fem_dense_field(const nrr_bm_fem *fem, const double *u, float *out_field, void *stream);
NRR_BM_API int nrr_bm_fem_dense_field_host(const nrr_bm_fem *fem, const double *u, float *out_field);
NRR_BM_API int nrr_bm_fem_destroy(nrr_bm_fem *fem);

/* Synchronises `stream` and returns NRR_E_DEVICE if a staged copy of a matching kernel enqueued on this thread since
 * the last check did not complete, NRR_E_BOUNDS if one saw a block leaving the volume (and clears the flag),
 * NRR_E_CUDA on a CUDA error, else NRR_OK. */
NRR_BM_API int nrr_bm_check_async_error(void *stream);

/*
 * Host-buffer forms (all pointers HOST memory; pinned memory makes the copies asynchronous).  They copy the
 * inputs to the device, run the same kernels as the device forms, copy the results back and synchronise.
 * nrr_bm_register_host = select + match of one volume pair in one call (both volumes uploaded once); this
 * is the end-to-end call bench.py times.  out_var / out_ncand may be NULL.
 */
NRR_BM_API int nrr_bm_select_blocks_host(const float *fixed, const int dims[3], const int block[3], const int stride[3],
                              double frac, const unsigned char *mask, int *out_blocks, int capacity,
                              int *out_n, double *out_var, int *out_ncand);
NRR_BM_API int nrr_bm_match_host(const float *fixed, const float *moving, const int dims[3], const int *blocks, int n,
                      const int block[3], const int window[3], int *out_disp, float *out_ncc);
NRR_BM_API int nrr_bm_register_host(const float *fixed, const float *moving, const int dims[3], const int block[3],
                         const int stride[3], const int window[3], double frac, const unsigned char *mask,
                         int *out_blocks, int capacity, int *out_n, int *out_disp, float *out_ncc);

/*
 * Instrumentation (no effect on results).
 *  nrr_bm_profile_enable(1): every later select/match call on this thread brackets its phases with CUDA
 *    events on the caller's stream.  nrr_bm_profile_read synchronises those events and returns the
 *    accumulated milliseconds and call counts since the last read, then resets them:
 *      ms[0] = selection kernels (statistics + radix select + compaction), ms[1] = moving-volume statistics
 *      (per-candidate normalisers), ms[2] = matching kernel alone, ms[3] = fixed-block records (the matching
 *      kernel's prep kernel);  calls[i] = number of timed launch groups.
 *  nrr_bm_launch_count(): kernels launched by this library on this thread since the last reset.
 *  nrr_bm_match_info: which matching kernel a (block, window, dims) triple dispatches to.
 *      info[0] = 2 pair kernel (two candidate rows per thread) / 1 one-row-per-thread kernel / 0 generic kernel,
 *      info[1] = threads per CTA, info[2] = dynamic shared memory bytes, info[3] = 1 if TMA staging is used,
 *      info[4] = candidates per block, info[5] = blocks per CTA.
 *  nrr_bm_fp32_peak: runs register-only FFMA / FFMA2 microbenchmarks on `stream`'s device and returns the best
 *      measured dense FP32 rate in TFLOP/s (the denominator context for the matching kernel's roofline).
 */
NRR_BM_API int nrr_bm_profile_enable(int on);
NRR_BM_API int nrr_bm_profile_read(double ms[4], int calls[4]);
NRR_BM_API long long nrr_bm_launch_count(int reset);
NRR_BM_API int nrr_bm_match_info(const int dims[3], const int block[3], const int window[3], int info[6]);
/*  nrr_bm_match_info_n: the same for a launch of n blocks (the pair kernel groups blocks into CTAs so that the last round
 *      of CTAs over the SMs is well filled; nrr_bm_match_info answers for a long block list). */
NRR_BM_API int nrr_bm_match_info_n(const int dims[3], const int block[3], const int window[3], int n, int info[6]);
NRR_BM_API int nrr_bm_fp32_peak(double *out_tflops, void *stream);
/*  nrr_bm_fp32_microbench: the FP32 microbenchmarks behind the matching kernel's design, TFLOP/s:
 *      out[0] FFMA register chain, out[1] FFMA register tile, out[2] FFMA2 (fma.rn.f32x2) packed x packed,
 *      out[3] FFMA2 scalar-broadcast x packed  (nrr_bm_fp32_peak = the best of these four);
 *      USEFUL TFLOP/s of three main-loop bodies on synthetic shared-memory data shaped like the 7^3 / +-5 search:
 *      out[4] one candidate row per thread with FFMA, out[5] two rows with FFMA, out[6] two rows with FFMA2. */
NRR_BM_API int nrr_bm_fp32_microbench(double out_tflops[7], void *stream);
/*  nrr_bm_pair_task_table: the host-built lane -> task table of the pair matching kernel for a cubic block and a
 *      window (wx == wy), one word per thread of a CTA: bit 31 = lane has a task, bit 30 = y-pair warp (the last
 *      candidate plane), bits 16..23 = block of the CTA's group, bits 8..15 = dy index, bits 0..7 = p: a z-pair task
 *      owns the rows (dy, dz = 2p) and (dy, 2p+1); a y-pair task owns (dy, dz = 2*wz) and, if p = 1, (dy+1, 2*wz).
 *      info[0] = threads per CTA (= words written), info[1] = blocks per CTA,
 *      info[2] = staged row pitch (floats), info[3] = staged rows per plane, info[4] = bytes between the unions of
 *      consecutive blocks in shared memory, info[5] = dynamic shared memory bytes.  No device needed. */
NRR_BM_API int nrr_bm_pair_task_table(const int block[3], const int window[3], unsigned int *out_table, int capacity,
                           int info[6]);

/* Tuning / experiment knobs (process-wide; results stay within the documented tolerances):
 *   "tie_band"      FP32 candidates within this NCC distance of the FP32 maximum are re-scored in FP64
 *                   (default 1e-4; 0 disables the re-score except for exact FP32 ties)
 *   "force_generic" != 0: always use the generic matching kernel
 *   "force_rows"    != 0: skip the pair kernel (one candidate row per thread instead)
 *   "disable_tma"   != 0: stage shared memory with plain loads instead of TMA
 *   "pair_blocks_per_cta"  > 0: blocks per CTA of the pair kernel (0 = the planner's choice)
 *   "plan_slabs"    z slabs of nrr_bm_plan_match_host's upload pipeline (default 4; 1 = upload, then compute)
 *   "boxstat_generic" / "select_generic" != 0: the runtime-shaped moving-statistics / selection kernels */
NRR_BM_API int nrr_bm_set_option(const char *name, double value);

NRR_BM_API const char *nrr_bm_last_error(void);
NRR_BM_API const char *nrr_bm_status_string(int status);
NRR_BM_API int nrr_bm_version(void);

#ifdef __cplusplus
}
#endif
#endif /* NRR_BM_H */
