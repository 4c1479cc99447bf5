/*
 * nrr_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * A plain, slow, obviously-correct CPU statement, in IEEE double precision, of what the block-matching
 * hot path of arxiv/paper_2308_10868 computes.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.  It shares no code, headers,
 * tables or helpers with paper_2308_10868_b200/ (the CUDA path) and neither includes the other.
 *
 * Image names follow BASELINE.json: "fixed" = the paper's floating / pre-operative
 * image (blocks are selected and cut here), "moving" = the paper's reference / intra-operative image (the
 * search window lives here).
 *
 * What each function follows:
 *   block variance, selection : PAPER.md:231-236 (section 3, "Sparse displacement vectors are obtained at
 *       the selected points ... where the variability in the intensities ... exceeds some threshold") and
 *       PAPER.md:376 (section 4.1 "Parallel feature selection": "computes the variance within a block",
 *       "selects F_s features with the highest variance", "0.5 + NFeatures x Fs blocks are selected").
 *   NCC                       : PAPER.md:243-246 (section 3 equation; garbled as printed, read as the
 *       standard Pearson form with both sums under the root -- DESIGN.md reading Q1).
 *   exhaustive search         : PAPER.md:236-243 and the listing PAPER.md:659-667 (section 4.3): for each
 *       block, every candidate block in the window, similarity, "find the maximum s and corresponding
 *       displacement".
 * Where the paper is silent the readings of DESIGN.md ("Readings of the paper", Q1-Q19) apply; the ones
 * with no pin in the paper are marked PARITY UNPINNED below and in DESIGN.md:
 *   - skip rule for candidates whose block leaves the moving volume (Q11)           PARITY UNPINNED
 *   - zero-variance block or candidate => NCC := 0 (Q12)                            PARITY UNPINNED
 *   - output order of the selected set = ascending candidate index (Q8)             PARITY UNPINNED
 *   - the pruning rule behind the paper's connectivity patterns (Q20)               PARITY UNPINNED
 *   - direction, interpolation and boundary rule of the dense-field warp (Q21)      PARITY UNPINNED
 * Everything else is pinned by tests/test_oracle_*.py (closed forms, numpy.corrcoef, translation
 * recovery, affine invariance, an independent naive evaluator in oracle/naive.py).
 *
 * Arithmetic: double, round-to-nearest, no FMA contraction (build with -ffp-contract=off), sums taken in
 * x-fastest order (x, then y, then z).  No blocking, fusion or reordering beyond the definitions.
 * OpenMP only distributes whole blocks over threads (blocks are independent); it never
 * changes the arithmetic of a block.
 *
 * Layout: voxel (x,y,z) of a volume with dims (nx,ny,nz) is at (z*ny + y)*nx + x.  Triples are (x,y,z).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define NRR_ORACLE_OK 0
#define NRR_ORACLE_E_ARG (-1)
#define NRR_ORACLE_E_CAPACITY (-2)
#define NRR_ORACLE_E_BOUNDS (-3)
#define NRR_ORACLE_E_NOMEM (-4)

static size_t vox(const int dims[3], int x, int y, int z)
{
    return ((size_t)z * (size_t)dims[1] + (size_t)y) * (size_t)dims[0] + (size_t)x;
}

/* Copy the block with origin o and extent b out of vol into buf, x fastest. */
static void gather_block(const float *vol, const int dims[3], const int o[3], const int b[3], double *buf)
{
    size_t k = 0;
    for (int z = 0; z < b[2]; ++z)
        for (int y = 0; y < b[1]; ++y)
            for (int x = 0; x < b[0]; ++x)
                buf[k++] = (double)vol[vox(dims, o[0] + x, o[1] + y, o[2] + z)];
}

/* Two-pass mean and sum of squared deviations of n values. */
static void mean_ss(const double *a, long n, double *mean, double *ss)
{
    double s = 0.0;
    for (long i = 0; i < n; ++i) s += a[i];
    double m = s / (double)n;
    double q = 0.0;
    for (long i = 0; i < n; ++i) {
        double d = a[i] - m;
        q += d * d;
    }
    *mean = m;
    *ss = q;
}

/* Population variance of n values ("computes the variance within a block"; population
 * rather than sample variance is reading Q7 -- the ranking is the same since |B| is constant). */
double nrr_oracle_variance(const double *a, long n)
{
    double m, q;
    mean_ss(a, n, &m, &q);
    return q / (double)n;
}

/* NCC of two equally long arrays (reading Q1):
 *     sum (a_i - abar)(b_i - bbar) / sqrt( sum (a_i - abar)^2 * sum (b_i - bbar)^2 )
 * Zero-variance argument => 0 (reading Q12, PARITY UNPINNED by the paper). */
double nrr_oracle_ncc(const double *a, const double *b, long n)
{
    double ma, ssa, mb, ssb;
    mean_ss(a, n, &ma, &ssa);
    mean_ss(b, n, &mb, &ssb);
    if (ssa == 0.0 || ssb == 0.0) return 0.0;
    double c = 0.0;
    for (long i = 0; i < n; ++i) c += (a[i] - ma) * (b[i] - mb);
    return c / sqrt(ssa * ssb);
}

/* float-input conveniences for the Python tests */
double nrr_oracle_variance_f32(const float *a, long n)
{
    double *t = (double *)malloc(sizeof(double) * (size_t)n);
    for (long i = 0; i < n; ++i) t[i] = (double)a[i];
    double v = nrr_oracle_variance(t, n);
    free(t);
    return v;
}

double nrr_oracle_ncc_f32(const float *a, const float *b, long n)
{
    double *t = (double *)malloc(sizeof(double) * (size_t)n * 2);
    for (long i = 0; i < n; ++i) { t[i] = (double)a[i]; t[n + i] = (double)b[i]; }
    double v = nrr_oracle_ncc(t, t + n, n);
    free(t);
    return v;
}

/* Count rule: "0.5 + NFeatures x Fs blocks are selected" => K = floor(0.5 + N*Fs) (Q6). */
int nrr_oracle_count(long n_candidates, double frac)
{
    return (int)floor(0.5 + (double)n_candidates * frac);
}

/* Grid extents of the stride grid (reading Q5): g_a = floor((n_a - B_a)/s_a) + 1, 0 if the block does
 * not fit. */
void nrr_oracle_grid(const int dims[3], const int block[3], const int stride[3], int g[3])
{
    for (int a = 0; a < 3; ++a)
        g[a] = (dims[a] >= block[a]) ? (dims[a] - block[a]) / stride[a] + 1 : 0;
}

typedef struct { double var; int q; int c[3]; } cand_t;

static int cmp_var_desc_q_asc(const void *pa, const void *pb)
{
    const cand_t *a = (const cand_t *)pa, *b = (const cand_t *)pb;
    if (a->var > b->var) return -1;
    if (a->var < b->var) return 1;
    return (a->q > b->q) - (a->q < b->q);
}

static int cmp_q_asc(const void *pa, const void *pb)
{
    const cand_t *a = (const cand_t *)pa, *b = (const cand_t *)pb;
    return (a->q > b->q) - (a->q < b->q);
}

/*
 * Variance-based block selection (readings Q5-Q10).
 *   candidates : stride grid from origin 0, blocks fully inside the volume, ascending linear grid order
 *                (x fastest); a grid position is a candidate iff mask == NULL or mask[centre] != 0 (Q9);
 *                variance is taken over the whole block regardless of the mask.
 *   keep       : the K = floor(0.5 + N*frac) candidates of largest variance, ties -> lower index (Q8).
 *   output     : block CENTRES (origin + (B-1)/2) in ascending candidate index; out_var (nullable) the
 *                variances in the same order; *out_ncand = N; *out_margin (nullable) = var of the K-th
 *                kept minus var of the best rejected candidate (inf if none rejected, nan if K == 0).
 * Returns 0, or NRR_ORACLE_E_CAPACITY if K > capacity (then *out_n = K and nothing else is written).
 */
int nrr_oracle_select(const float *fixed, const int dims[3], const int block[3], const int stride[3],
                      double frac, const unsigned char *mask, int *out_centres, int capacity,
                      int *out_n, double *out_var, int *out_ncand, double *out_margin)
{
    for (int a = 0; a < 3; ++a)
        if (dims[a] < 1 || block[a] < 1 || (block[a] & 1) == 0 || stride[a] < 1) return NRR_ORACLE_E_ARG;
    if (!(frac > 0.0 && frac <= 1.0)) return NRR_ORACLE_E_ARG;
    int g[3];
    nrr_oracle_grid(dims, block, stride, g);
    size_t ngrid = (size_t)g[0] * (size_t)g[1] * (size_t)g[2];
    long nb = (long)block[0] * block[1] * block[2];
    cand_t *cand = (cand_t *)malloc(sizeof(cand_t) * (ngrid ? ngrid : 1));
    double *buf = (double *)malloc(sizeof(double) * (size_t)nb);
    if (!cand || !buf) { free(cand); free(buf); return NRR_ORACLE_E_NOMEM; }
    int n = 0;
    for (int k = 0; k < g[2]; ++k)
        for (int j = 0; j < g[1]; ++j)
            for (int i = 0; i < g[0]; ++i) {
                int o[3] = { i * stride[0], j * stride[1], k * stride[2] };
                int c[3] = { o[0] + (block[0] - 1) / 2, o[1] + (block[1] - 1) / 2, o[2] + (block[2] - 1) / 2 };
                if (mask && mask[vox(dims, c[0], c[1], c[2])] == 0) continue;
                gather_block(fixed, dims, o, block, buf);
                cand[n].var = nrr_oracle_variance(buf, nb);
                cand[n].q = n;
                cand[n].c[0] = c[0]; cand[n].c[1] = c[1]; cand[n].c[2] = c[2];
                ++n;
            }
    free(buf);
    int K = nrr_oracle_count(n, frac);
    if (K > n) K = n;
    *out_n = K;
    if (out_ncand) *out_ncand = n;
    if (K > capacity) { free(cand); return NRR_ORACLE_E_CAPACITY; }
    qsort(cand, (size_t)n, sizeof(cand_t), cmp_var_desc_q_asc);
    if (out_margin) {
        if (K == 0) *out_margin = NAN;
        else if (K == n) *out_margin = INFINITY;
        else *out_margin = cand[K - 1].var - cand[K].var;
    }
    qsort(cand, (size_t)K, sizeof(cand_t), cmp_q_asc);
    for (int t = 0; t < K; ++t) {
        out_centres[3 * t + 0] = cand[t].c[0];
        out_centres[3 * t + 1] = cand[t].c[1];
        out_centres[3 * t + 2] = cand[t].c[2];
        if (out_var) out_var[t] = cand[t].var;
    }
    free(cand);
    return NRR_ORACLE_OK;
}

/*
 * Selection with the connectivity pattern ("The method also uses a connectivity pattern to avoid
 * selecting blocks that are too close to each other ... Three simplex patterns are available: vertex (26
 * connectivity), edge (18 connectivity), face (6 connectivity)").  The paper names the patterns but not the
 * pruning algorithm; reading Q20, PARITY UNPINNED by the paper:
 *   candidates, variances, N and K = floor(0.5 + N*frac) exactly as in nrr_oracle_select;
 *   walk the candidates by (variance descending, candidate index ascending); KEEP a candidate iff none of its
 *   neighbours ON THE CANDIDATE GRID (grid offsets (di,dj,dk) in {-1,0,1}^3 \ {0} with |di|+|dj|+|dk| <= 1 for
 *   connectivity 6, <= 2 for 18, <= 3 for 26) has been kept already; stop once K are kept or the list ends;
 *   output the kept centres in ascending candidate index.  connectivity 0 = no pruning.
 * With stride 1 the grid neighbours are the voxel neighbours of the block centre (the paper's setting: every
 * intracranial voxel is a feature candidate).  Out-of-mask grid positions are not candidates and block nothing.
 */
int nrr_oracle_select_pruned(const float *fixed, const int dims[3], const int block[3], const int stride[3],
                             double frac, const unsigned char *mask, int connectivity, int *out_centres,
                             int capacity, int *out_n, double *out_var, int *out_ncand)
{
    for (int a = 0; a < 3; ++a)
        if (dims[a] < 1 || block[a] < 1 || (block[a] & 1) == 0 || stride[a] < 1) return NRR_ORACLE_E_ARG;
    if (!(frac > 0.0 && frac <= 1.0)) return NRR_ORACLE_E_ARG;
    if (connectivity != 0 && connectivity != 6 && connectivity != 18 && connectivity != 26) return NRR_ORACLE_E_ARG;
    const int reach = connectivity == 6 ? 1 : connectivity == 18 ? 2 : connectivity == 26 ? 3 : 0;
    int g[3];
    nrr_oracle_grid(dims, block, stride, g);
    size_t ngrid = (size_t)g[0] * (size_t)g[1] * (size_t)g[2];
    long nb = (long)block[0] * block[1] * block[2];
    cand_t *cand = (cand_t *)malloc(sizeof(cand_t) * (ngrid ? ngrid : 1));
    int *gpos = (int *)malloc(sizeof(int) * 3 * (ngrid ? ngrid : 1));          /* grid coordinates per candidate */
    unsigned char *kept = (unsigned char *)calloc(ngrid ? ngrid : 1, 1);       /* per GRID position */
    double *buf = (double *)malloc(sizeof(double) * (size_t)nb);
    if (!cand || !gpos || !kept || !buf) { free(cand); free(gpos); free(kept); free(buf); return NRR_ORACLE_E_NOMEM; }
    int n = 0;
    for (int k = 0; k < g[2]; ++k)
        for (int j = 0; j < g[1]; ++j)
            for (int i = 0; i < g[0]; ++i) {
                int o[3] = { i * stride[0], j * stride[1], k * stride[2] };
                int c[3] = { o[0] + (block[0] - 1) / 2, o[1] + (block[1] - 1) / 2, o[2] + (block[2] - 1) / 2 };
                if (mask && mask[vox(dims, c[0], c[1], c[2])] == 0) continue;
                gather_block(fixed, dims, o, block, buf);
                cand[n].var = nrr_oracle_variance(buf, nb);
                cand[n].q = n;
                cand[n].c[0] = c[0]; cand[n].c[1] = c[1]; cand[n].c[2] = c[2];
                gpos[3 * n + 0] = i; gpos[3 * n + 1] = j; gpos[3 * n + 2] = k;
                ++n;
            }
    free(buf);
    int K = nrr_oracle_count(n, frac);
    if (K > n) K = n;
    if (out_ncand) *out_ncand = n;
    qsort(cand, (size_t)n, sizeof(cand_t), cmp_var_desc_q_asc);
    int nk = 0;                                   /* kept candidates are moved to the front of cand[] */
    for (int t = 0; t < n && nk < K; ++t) {
        const int *gp = gpos + 3 * cand[t].q;
        int blocked = 0;
        for (int dk = -1; dk <= 1 && !blocked; ++dk)
            for (int dj = -1; dj <= 1 && !blocked; ++dj)
                for (int di = -1; di <= 1 && !blocked; ++di) {
                    int m = abs(di) + abs(dj) + abs(dk);
                    if (m == 0 || m > reach) continue;
                    int i = gp[0] + di, j = gp[1] + dj, k = gp[2] + dk;
                    if (i < 0 || j < 0 || k < 0 || i >= g[0] || j >= g[1] || k >= g[2]) continue;
                    if (kept[((size_t)k * g[1] + j) * g[0] + i]) blocked = 1;
                }
        if (blocked) continue;
        kept[((size_t)gp[2] * g[1] + gp[1]) * g[0] + gp[0]] = 1;
        cand[nk++] = cand[t];
    }
    *out_n = nk;
    if (nk > capacity) { free(cand); free(gpos); free(kept); return NRR_ORACLE_E_CAPACITY; }
    qsort(cand, (size_t)nk, sizeof(cand_t), cmp_q_asc);
    for (int t = 0; t < nk; ++t) {
        out_centres[3 * t + 0] = cand[t].c[0];
        out_centres[3 * t + 1] = cand[t].c[1];
        out_centres[3 * t + 2] = cand[t].c[2];
        if (out_var) out_var[t] = cand[t].var;
    }
    free(cand); free(gpos); free(kept);
    return NRR_ORACLE_OK;
}

/*
 * Exhaustive NCC block matching (listing PAPER.md:659-667; readings Q11-Q15).
 * For each centre c (block origin o = c - (B-1)/2 in the fixed volume):
 *   for dz, dy, dx ascending (linear candidate index ((dz+rz)(2ry+1) + (dy+ry))(2rx+1) + (dx+rx)):
 *       skip d if the block at o+d leaves the moving volume (Q11)
 *       ncc = NCC(fixed block at o, moving block at o+d)
 *       strictly greater than the best so far => new best (so equal maxima keep the lowest index, Q13)
 *   out_disp = d*, out_ncc = best, out_gap = best - second largest value (inf if one candidate only),
 *   out_nvalid = number of candidates evaluated.
 * Sign convention (Q15): fixed(p + v) ~ moving(p + d + v).  Units: voxels.
 * nthreads <= 0: OpenMP default.  Returns 0 or NRR_ORACLE_E_BOUNDS if a block leaves the volume.
 */
int nrr_oracle_match(const float *fixed, const float *moving, const int dims[3], const int *centres,
                     int n, const int block[3], const int window[3], int *out_disp, double *out_ncc,
                     double *out_gap, int *out_nvalid, int nthreads)
{
    for (int a = 0; a < 3; ++a)
        if (dims[a] < 1 || block[a] < 1 || (block[a] & 1) == 0 || window[a] < 0) return NRR_ORACLE_E_ARG;
    long nb = (long)block[0] * block[1] * block[2];
    for (int b = 0; b < n; ++b)
        for (int a = 0; a < 3; ++a) {
            int o = centres[3 * b + a] - (block[a] - 1) / 2;
            if (o < 0 || o + block[a] > dims[a]) return NRR_ORACLE_E_BOUNDS;
        }
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
    int err = 0;
#pragma omp parallel
    {
        double *fb = (double *)malloc(sizeof(double) * (size_t)nb);
        double *mb = (double *)malloc(sizeof(double) * (size_t)nb);
        if (!fb || !mb) {
#pragma omp atomic write
            err = 1;
        }
#pragma omp for schedule(dynamic, 4)
        for (int b = 0; b < n; ++b) {
            if (!fb || !mb) continue;
            int o[3];
            for (int a = 0; a < 3; ++a) o[a] = centres[3 * b + a] - (block[a] - 1) / 2;
            gather_block(fixed, dims, o, block, fb);
            double best = -INFINITY, second = -INFINITY;
            int bd[3] = { 0, 0, 0 };
            int nvalid = 0;
            for (int dz = -window[2]; dz <= window[2]; ++dz)
                for (int dy = -window[1]; dy <= window[1]; ++dy)
                    for (int dx = -window[0]; dx <= window[0]; ++dx) {
                        int p[3] = { o[0] + dx, o[1] + dy, o[2] + dz };
                        if (p[0] < 0 || p[1] < 0 || p[2] < 0 || p[0] + block[0] > dims[0] ||
                            p[1] + block[1] > dims[1] || p[2] + block[2] > dims[2])
                            continue;
                        gather_block(moving, dims, p, block, mb);
                        double s = nrr_oracle_ncc(fb, mb, nb);
                        ++nvalid;
                        if (s > best) {
                            second = best;
                            best = s;
                            bd[0] = dx; bd[1] = dy; bd[2] = dz;
                        } else if (s > second) {
                            second = s;
                        }
                    }
            out_disp[3 * b + 0] = bd[0];
            out_disp[3 * b + 1] = bd[1];
            out_disp[3 * b + 2] = bd[2];
            out_ncc[b] = best;
            if (out_gap) out_gap[b] = (nvalid > 1) ? best - second : INFINITY;
            if (out_nvalid) out_nvalid[b] = nvalid;
        }
        free(fb);
        free(mb);
    }
    return err ? NRR_ORACLE_E_NOMEM : NRR_ORACLE_OK;
}

/* NCC of one (block, displacement) pair -- lets tests sample single candidates at full problem sizes.
 * Returns nan if the candidate is skipped by the rule above. */
double nrr_oracle_ncc_at(const float *fixed, const float *moving, const int dims[3], const int centre[3],
                         const int block[3], const int d[3])
{
    long nb = (long)block[0] * block[1] * block[2];
    int o[3], p[3];
    for (int a = 0; a < 3; ++a) {
        o[a] = centre[a] - (block[a] - 1) / 2;
        p[a] = o[a] + d[a];
        if (o[a] < 0 || o[a] + block[a] > dims[a]) return NAN;
        if (p[a] < 0 || p[a] + block[a] > dims[a]) return NAN;
    }
    double *fb = (double *)malloc(sizeof(double) * (size_t)nb * 2);
    double *mb = fb + nb;
    gather_block(fixed, dims, o, block, fb);
    gather_block(moving, dims, p, block, mb);
    double s = nrr_oracle_ncc(fb, mb, nb);
    free(fb);
    return s;
}

/*
 * Warp of an image by a dense displacement field (the registration derives a "dense
 * deformation field that defines transformation for each point in the image space", which is then applied to the
 * pre-operative image; the APBNRR loop of PAPER.md:286 re-registers the warped image).  The paper gives no
 * formula; reading Q21, PARITY UNPINNED by the paper: backward warp on the output grid with trilinear
 * interpolation and edge clamping,
 *     out(p) = T[image](p + v(p)),   v(p) = (field[0][p], field[1][p], field[2][p])  in voxels, (x, y, z) order,
 * where the sample position is clamped to [0, n_a - 1] per axis and T interpolates linearly along x, then y,
 * then z between the two neighbouring voxels.  Arithmetic in double; the result is rounded to float once.
 */
int nrr_oracle_warp(const float *image, const int dims[3], const float *field, float *out)
{
    for (int a = 0; a < 3; ++a)
        if (dims[a] < 1) return NRR_ORACLE_E_ARG;
    const size_t nvox = (size_t)dims[0] * dims[1] * dims[2];
    for (int z = 0; z < dims[2]; ++z)
        for (int y = 0; y < dims[1]; ++y)
            for (int x = 0; x < dims[0]; ++x) {
                const size_t p = vox(dims, x, y, z);
                const int pos[3] = { x, y, z };
                int i0[3], i1[3];
                double t[3];
                for (int a = 0; a < 3; ++a) {
                    double s = (double)pos[a] + (double)field[(size_t)a * nvox + p];
                    if (s < 0.0) s = 0.0;
                    if (s > (double)(dims[a] - 1)) s = (double)(dims[a] - 1);
                    double f = floor(s);
                    i0[a] = (int)f;
                    i1[a] = i0[a] + 1 < dims[a] ? i0[a] + 1 : i0[a];
                    t[a] = s - f;
                }
                double c[2][2];
                for (int kz = 0; kz < 2; ++kz)
                    for (int ky = 0; ky < 2; ++ky) {
                        const int zz = kz ? i1[2] : i0[2], yy = ky ? i1[1] : i0[1];
                        const double a0 = (double)image[vox(dims, i0[0], yy, zz)];
                        const double a1 = (double)image[vox(dims, i1[0], yy, zz)];
                        c[kz][ky] = a0 + t[0] * (a1 - a0);
                    }
                const double c0 = c[0][0] + t[1] * (c[0][1] - c[0][0]);
                const double c1 = c[1][0] + t[1] * (c[1][1] - c[1][0]);
                out[p] = (float)(c0 + t[2] * (c1 - c0));
            }
    return NRR_ORACLE_OK;
}


int nrr_oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
