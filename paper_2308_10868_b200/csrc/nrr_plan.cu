// nrr_plan.cu -- the boundary split along the paper's timeline (include/nrr_bm.h "PLANS") and the parameter
// sweep in one launch sequence ("PARAMETER SWEEP").  Host-side orchestration only: every step of the path runs in
// the kernels of nrr_select.cu / nrr_boxstat.cu / nrr_match*.cu.
//
//   pre-operative: selection S1-S3, the fixed-block records of the matching kernel, scratch;
//   intra-operative: moving-volume normalisers M2, matching M1/M3-M5.
#include <math.h>
#include <string.h>

#include <algorithm>
#include <map>
#include <tuple>
#include <vector>

#include "nrr_internal.cuh"

namespace nrr {
extern int g_plan_slabs;
int g_plan_slabs = 4;      // z slabs of the host form's upload pipeline (option "plan_slabs")
}

using namespace nrr;

struct nrr_bm_plan {
    unsigned int magic = 0;
    int device = 0;
    Int3 dims{}, block{}, stride{}, window{};
    double frac = 0.0;
    int connectivity = 0;
    int n = 0, ncand = 0;
    bool owns_fixed = false;
    const float *fixed = nullptr;      // device
    int *blocks = nullptr;             // device [n][3]
    double *var = nullptr;             // device [n]
    float *records = nullptr;          // device, match_records_bytes(...) (NULL: the kernel keeps no records)
    float *inv_sd = nullptr;           // device [nvox], rewritten by every match call
    // host form
    float *moving_dev = nullptr;       // device [nvox]
    int *disp_dev = nullptr;           // device [n][3]
    float *ncc_dev = nullptr;          // device [n]
    cudaStream_t copy_stream = nullptr;
    std::vector<cudaEvent_t> slab_events;
    std::vector<int> blocks_host;      // [n][3]
    std::vector<double> var_host;      // [n]
};

namespace {

constexpr unsigned int kPlanMagic = 0x4e525250u;      // "NRRP"

Int3 i3(const int v[3]) { return Int3{v[0], v[1], v[2]}; }

int check_window(const int window[3])
{
    if (!window) return api_fail(NRR_E_NULL, "window is NULL");
    for (int a = 0; a < 3; ++a)
        if (window[a] < 0) return api_fail(NRR_E_WINDOW, "window[%d] = %d < 0", a, window[a]);
    return NRR_OK;
}

Int3 grid_of(Int3 dims, Int3 block, Int3 stride)
{
    return Int3{(dims.x - block.x) / stride.x + 1, (dims.y - block.y) / stride.y + 1, (dims.z - block.z) / stride.z + 1};
}

int plan_ok(const nrr_bm_plan *p)
{
    if (!p || p->magic != kPlanMagic) return api_fail(NRR_E_ARG, "not a live nrr_bm_plan");
    int dev = 0;
    NRR_CUDA(cudaGetDevice(&dev));
    if (dev != p->device) return api_fail(NRR_E_ARG, "the plan belongs to device %d, the current device is %d", p->device, dev);
    return NRR_OK;
}

void plan_free(nrr_bm_plan *p)
{
    if (!p) return;
    if (p->owns_fixed && p->fixed) cudaFree((void *)p->fixed);
    if (p->blocks) cudaFree(p->blocks);
    if (p->var) cudaFree(p->var);
    if (p->records) cudaFree(p->records);
    if (p->inv_sd) cudaFree(p->inv_sd);
    if (p->moving_dev) cudaFree(p->moving_dev);
    if (p->disp_dev) cudaFree(p->disp_dev);
    if (p->ncc_dev) cudaFree(p->ncc_dev);
    for (cudaEvent_t e : p->slab_events) cudaEventDestroy(e);
    p->magic = 0;
    delete p;
}

// Selection + records on `stream`; fills the plan.  `fixed` / `mask`: device.
int plan_build(nrr_bm_plan *p, const float *fixed, const unsigned char *mask, cudaStream_t stream)
{
    unsigned int *err_flag = nullptr;
    void *pinned = nullptr;
    int rc = api_thread_state(&err_flag, &pinned);
    if (rc) return rc;
    MatchPlan mp;
    if ((rc = match_plan(p->dims, p->block, p->window, nullptr, fixed, &mp))) return rc;      // NRR_E_SMEM for impossible shapes
    const Int3 g = grid_of(p->dims, p->block, p->stride);
    const long long ngrid = (long long)g.x * g.y * g.z;
    if (ngrid > 0x7fffffffll) return api_fail(NRR_E_DIMS, "stride grid has %lld positions (limit 2^31-1)", ngrid);
    const long long kmax = api_capacity_bound(ngrid, p->frac);
    const int cap = (int)(kmax > 0 ? kmax : 1);
    // selection into call scratch of the bound's size; the plan keeps exact-size copies
    AsyncScratch sel_buf(stream), blk_buf(stream), var_buf(stream);
    NRR_CUDA(sel_buf.alloc(select_scratch_bytes(ngrid)));
    NRR_CUDA(blk_buf.alloc((size_t)cap * 3 * sizeof(int)));
    NRR_CUDA(var_buf.alloc((size_t)cap * sizeof(double)));
    SelectState *st = nullptr;
    profile_begin(0, stream);
    rc = select_enqueue(fixed, p->dims, p->block, p->stride, g, p->frac, mask, (int *)blk_buf.p, cap, (double *)var_buf.p,
                        sel_buf.p, &st, stream, p->connectivity, (SelectState *)((char *)pinned + 3072));
    profile_end(0, stream);
    if (rc) return rc;
    SelectState *h = (SelectState *)pinned;
    NRR_CUDA(cudaMemcpyAsync(h, st, sizeof(SelectState), cudaMemcpyDeviceToHost, stream));
    NRR_CUDA(cudaStreamSynchronize(stream));
    p->n = (int)h->k;
    p->ncand = (int)h->n_candidates;
    if (p->n > cap) return api_fail(NRR_E_CAPACITY, "K = %d exceeds the library's own bound %d", p->n, cap);
    const size_t n1 = (size_t)(p->n > 0 ? p->n : 1);
    NRR_CUDA(cudaMalloc((void **)&p->blocks, n1 * 3 * sizeof(int)));
    NRR_CUDA(cudaMalloc((void **)&p->var, n1 * sizeof(double)));
    p->blocks_host.assign((size_t)p->n * 3, 0);
    p->var_host.assign((size_t)p->n, 0.0);
    if (p->n > 0) {
        NRR_CUDA(cudaMemcpyAsync(p->blocks, blk_buf.p, (size_t)p->n * 3 * sizeof(int), cudaMemcpyDeviceToDevice, stream));
        NRR_CUDA(cudaMemcpyAsync(p->var, var_buf.p, (size_t)p->n * sizeof(double), cudaMemcpyDeviceToDevice, stream));
        NRR_CUDA(cudaMemcpyAsync(p->blocks_host.data(), blk_buf.p, (size_t)p->n * 3 * sizeof(int), cudaMemcpyDeviceToHost, stream));
        NRR_CUDA(cudaMemcpyAsync(p->var_host.data(), var_buf.p, (size_t)p->n * sizeof(double), cudaMemcpyDeviceToHost, stream));
    }
    const size_t nvox = (size_t)p->dims.x * p->dims.y * p->dims.z;
    NRR_CUDA(cudaMalloc((void **)&p->inv_sd, nvox * sizeof(float)));
    p->fixed = fixed;
    const size_t rec_bytes = match_records_bytes(p->block, p->window, p->n);
    if (rec_bytes > 0) {
        NRR_CUDA(cudaMalloc((void **)&p->records, rec_bytes));
        MatchCall c;
        c.fixed = fixed; c.dims = p->dims; c.block = p->block; c.window = p->window; c.blocks = p->blocks; c.n = p->n;
        c.records = p->records; c.phase = kMatchPrepOnly; c.err_flag = err_flag; c.stream = stream;
        if ((rc = match_enqueue(c))) return rc;
    }
    NRR_CUDA(cudaStreamSynchronize(stream));
    return NRR_OK;
}

int plan_create_common(const float *fixed, const int dims[3], const int block[3], const int stride[3], const int window[3],
                       double frac, const unsigned char *mask, int connectivity, cudaStream_t stream, bool host_inputs,
                       nrr_bm_plan **out_plan)
{
    if (!out_plan) return api_fail(NRR_E_NULL, "out_plan is NULL");
    *out_plan = nullptr;
    int rc = api_check_select_args(fixed, dims, block, stride, frac);
    if (rc) return rc;
    if ((rc = check_window(window))) return rc;
    if (connectivity != 0 && connectivity != 6 && connectivity != 18 && connectivity != 26)
        return api_fail(NRR_E_ARG, "connectivity = %d (0, 6, 18 or 26)", connectivity);
    nrr_bm_plan *p = new nrr_bm_plan();
    p->magic = kPlanMagic;
    p->dims = i3(dims); p->block = i3(block); p->stride = i3(stride); p->window = i3(window);
    p->frac = frac; p->connectivity = connectivity;
    if (cudaGetDevice(&p->device) != cudaSuccess) { plan_free(p); return api_fail(NRR_E_CUDA, "no CUDA device"); }
    const size_t nvox = (size_t)dims[0] * dims[1] * dims[2];
    const float *d_fixed = fixed;
    unsigned char *d_mask = nullptr;
    auto fail_with = [&](int code) { if (d_mask) cudaFree(d_mask); plan_free(p); return code; };
    if (host_inputs) {
        if ((rc = api_host_stream(&stream))) return fail_with(rc);
        float *df = nullptr;
        if (cudaMalloc((void **)&df, nvox * sizeof(float)) != cudaSuccess) return fail_with(api_fail(NRR_E_CUDA, "cudaMalloc of the fixed volume failed"));
        p->fixed = df; p->owns_fixed = true; d_fixed = df;
        if (cudaMemcpyAsync(df, fixed, nvox * sizeof(float), cudaMemcpyHostToDevice, stream) != cudaSuccess)
            return fail_with(api_fail(NRR_E_CUDA, "upload of the fixed volume failed"));
        if (mask) {
            if (cudaMalloc((void **)&d_mask, nvox) != cudaSuccess ||
                cudaMemcpyAsync(d_mask, mask, nvox, cudaMemcpyHostToDevice, stream) != cudaSuccess)
                return fail_with(api_fail(NRR_E_CUDA, "upload of the mask failed"));
        }
    }
    rc = plan_build(p, d_fixed, host_inputs ? d_mask : mask, stream);
    if (rc) return fail_with(rc);
    if (d_mask) { cudaFree(d_mask); d_mask = nullptr; }      // the stream was synchronised by plan_build
    *out_plan = p;
    return NRR_OK;
}

// M2 + matching of blocks [first, first + count) on `stream`; the moving volume must have landed up to (exclusive)
// plane z_ready for everything these blocks read, which the callers guarantee.
int plan_enqueue(nrr_bm_plan *p, const float *moving, int first, int count, int zo_lo, int zo_hi, int *out_disp,
                 float *out_ncc, cudaStream_t stream)
{
    unsigned int *err_flag = nullptr;
    int rc = api_thread_state(&err_flag, nullptr);
    if (rc) return rc;
    profile_begin(1, stream);
    rc = boxstat_enqueue_range(moving, p->dims, p->block, p->inv_sd, zo_lo, zo_hi, stream);
    profile_end(1, stream);
    if (rc || count <= 0) return rc;
    const size_t rec_stride = p->records ? match_records_bytes(p->block, p->window, 1) : 0;
    MatchCall c;
    c.fixed = p->fixed; c.moving = moving; c.inv_sd = p->inv_sd; c.dims = p->dims; c.block = p->block; c.window = p->window;
    c.blocks = p->blocks + 3 * (size_t)first; c.n = count;
    c.out_disp = out_disp + 3 * (size_t)first; c.out_ncc = out_ncc + first;
    c.err_flag = err_flag; c.stream = stream;
    if (p->records) {
        c.records = (float *)((char *)p->records + (size_t)first * rec_stride);
        c.phase = kMatchKernelOnly;
    }
    return match_enqueue(c);
}

}  // namespace

extern "C" {

int nrr_bm_capacity_bound(const int dims[3], const int block[3], const int stride[3], double frac, int *out_grid,
                          int *out_bound)
{
    int rc = api_check_dims_block(dims, block);
    if (rc) return rc;
    if (!stride) return api_fail(NRR_E_NULL, "stride is NULL");
    for (int a = 0; a < 3; ++a)
        if (stride[a] < 1) return api_fail(NRR_E_STRIDE, "stride[%d] = %d < 1", a, stride[a]);
    if (!(frac > 0.0 && frac <= 1.0)) return api_fail(NRR_E_FRAC, "frac = %g outside (0, 1]", frac);
    const Int3 g = grid_of(i3(dims), i3(block), i3(stride));
    const long long ngrid = (long long)g.x * g.y * g.z;
    if (ngrid > 0x7fffffffll) return api_fail(NRR_E_DIMS, "stride grid has %lld positions (limit 2^31-1)", ngrid);
    if (out_grid) *out_grid = (int)ngrid;
    if (out_bound) *out_bound = (int)api_capacity_bound(ngrid, frac);
    return NRR_OK;
}

int nrr_bm_plan_create(const float *fixed, const int dims[3], const int block[3], const int stride[3],
                       const int window[3], double frac, const unsigned char *mask, int connectivity, void *stream,
                       nrr_bm_plan **out_plan)
{
    return plan_create_common(fixed, dims, block, stride, window, frac, mask, connectivity, (cudaStream_t)stream, false, out_plan);
}

int nrr_bm_plan_create_host(const float *fixed, const int dims[3], const int block[3], const int stride[3],
                            const int window[3], double frac, const unsigned char *mask, int connectivity,
                            nrr_bm_plan **out_plan)
{
    return plan_create_common(fixed, dims, block, stride, window, frac, mask, connectivity, nullptr, true, out_plan);
}

int nrr_bm_plan_info(const nrr_bm_plan *plan, int *out_n, int *out_ncand)
{
    if (!plan || plan->magic != kPlanMagic) return api_fail(NRR_E_ARG, "not a live nrr_bm_plan");
    if (out_n) *out_n = plan->n;
    if (out_ncand) *out_ncand = plan->ncand;
    return NRR_OK;
}

int nrr_bm_plan_blocks_host(const nrr_bm_plan *plan, int *out_blocks, double *out_var)
{
    if (!plan || plan->magic != kPlanMagic) return api_fail(NRR_E_ARG, "not a live nrr_bm_plan");
    if (plan->n > 0 && !out_blocks) return api_fail(NRR_E_NULL, "out_blocks is NULL");
    if (plan->n > 0) memcpy(out_blocks, plan->blocks_host.data(), (size_t)plan->n * 3 * sizeof(int));
    if (plan->n > 0 && out_var) memcpy(out_var, plan->var_host.data(), (size_t)plan->n * sizeof(double));
    return NRR_OK;
}

int nrr_bm_plan_blocks(const nrr_bm_plan *plan, int *out_blocks, double *out_var, void *stream)
{
    int rc = plan_ok(plan);
    if (rc) return rc;
    if (plan->n > 0 && !out_blocks) return api_fail(NRR_E_NULL, "out_blocks is NULL");
    if (plan->n == 0) return NRR_OK;
    NRR_CUDA(cudaMemcpyAsync(out_blocks, plan->blocks, (size_t)plan->n * 3 * sizeof(int), cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
    if (out_var) NRR_CUDA(cudaMemcpyAsync(out_var, plan->var, (size_t)plan->n * sizeof(double), cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
    return NRR_OK;
}

const int *nrr_bm_plan_blocks_device(const nrr_bm_plan *plan)
{
    if (!plan || plan->magic != kPlanMagic) { api_fail(NRR_E_ARG, "not a live nrr_bm_plan"); return nullptr; }
    return plan->blocks;
}

int nrr_bm_plan_match_range(nrr_bm_plan *plan, const float *moving, int first, int count, int *out_disp, float *out_ncc,
                            void *stream)
{
    int rc = plan_ok(plan);
    if (rc) return rc;
    if (!moving) return api_fail(NRR_E_NULL, "moving is NULL");
    if (first < 0 || count < 0 || first > plan->n || count > plan->n - first)
        return api_fail(NRR_E_ARG, "block range [%d, %d + %d) outside [0, %d]", first, first, count, plan->n);
    if (count > 0 && (!out_disp || !out_ncc)) return api_fail(NRR_E_NULL, "out_disp/out_ncc is NULL");
    if (count == 0) return NRR_OK;
    // normalisers only for the planes this slice of the (z-major) block list can reach
    const int bz = plan->block.z, rz = plan->window.z;
    const int oz_first = plan->blocks_host[3 * (size_t)first + 2] - (bz - 1) / 2;
    const int oz_last = plan->blocks_host[3 * (size_t)(first + count - 1) + 2] - (bz - 1) / 2;
    return plan_enqueue(plan, moving, first, count, oz_first - rz, oz_last + rz + 1, out_disp, out_ncc, (cudaStream_t)stream);
}

int nrr_bm_plan_match(nrr_bm_plan *plan, const float *moving, int *out_disp, float *out_ncc, void *stream)
{
    int rc = plan_ok(plan);
    if (rc) return rc;
    return nrr_bm_plan_match_range(plan, moving, 0, plan->n, out_disp, out_ncc, stream);
}

int nrr_bm_plan_match_host(nrr_bm_plan *plan, const float *moving, int *out_disp, float *out_ncc)
{
    int rc = plan_ok(plan);
    if (rc) return rc;
    if (!moving) return api_fail(NRR_E_NULL, "moving is NULL");
    const int n = plan->n;
    if (n > 0 && (!out_disp || !out_ncc)) return api_fail(NRR_E_NULL, "out_disp/out_ncc is NULL");
    if (n == 0) return NRR_OK;
    cudaStream_t s;
    if ((rc = api_host_stream(&s))) return rc;
    const Int3 dims = plan->dims;
    const size_t plane = (size_t)dims.x * dims.y, nvox = plane * dims.z;
    if (!plan->moving_dev) {
        NRR_CUDA(cudaMalloc((void **)&plan->moving_dev, nvox * sizeof(float)));
        NRR_CUDA(cudaMalloc((void **)&plan->disp_dev, (size_t)n * 3 * sizeof(int)));
        NRR_CUDA(cudaMalloc((void **)&plan->ncc_dev, (size_t)n * sizeof(float)));
        NRR_CUDA(cudaStreamCreateWithFlags(&plan->copy_stream, cudaStreamNonBlocking));
    }
    const int bz = plan->block.z, rz = plan->window.z, nzo = dims.z - bz + 1;
    int nslab = g_plan_slabs < 1 ? 1 : g_plan_slabs;
    if (nslab > dims.z) nslab = dims.z;
    while ((int)plan->slab_events.size() < nslab) {
        cudaEvent_t e = nullptr;
        NRR_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        plan->slab_events.push_back(e);
    }
    // Slab i ends (exclusive) at plane z_end.  Once it has landed, the normalisers of every block origin whose block
    // lies below z_end are due, and so is the matching of every block whose whole window union lies below z_end (the
    // union is clipped at the volume's end, where the hardware zero-fills).  The block list is z-major, so these are
    // contiguous ranges that only grow.
    int z_done = 0, zo_done = 0, b_done = 0;
    for (int i = 0; i < nslab; ++i) {
        const int z_end = (int)(((long long)dims.z * (i + 1)) / nslab);
        if (z_end <= z_done) continue;
        NRR_CUDA(cudaMemcpyAsync(plan->moving_dev + (size_t)z_done * plane, moving + (size_t)z_done * plane,
                                 (size_t)(z_end - z_done) * plane * sizeof(float), cudaMemcpyHostToDevice, plan->copy_stream));
        NRR_CUDA(cudaEventRecord(plan->slab_events[(size_t)i], plan->copy_stream));
        NRR_CUDA(cudaStreamWaitEvent(s, plan->slab_events[(size_t)i], 0));
        z_done = z_end;
        int zo_hi = z_end - bz + 1;                      // origins whose block ends at or before z_end
        if (zo_hi > nzo) zo_hi = nzo;
        if (zo_hi < zo_done) zo_hi = zo_done;
        int b_hi = b_done;
        while (b_hi < n) {
            const int oz = plan->blocks_host[3 * (size_t)b_hi + 2] - (bz - 1) / 2;
            int top = oz + rz + bz;                      // exclusive end of the window union along z
            if (top > dims.z) top = dims.z;
            if (top > z_end) break;
            ++b_hi;
        }
        rc = plan_enqueue(plan, plan->moving_dev, b_done, b_hi - b_done, zo_done, zo_hi, plan->disp_dev, plan->ncc_dev, s);
        if (rc) return rc;
        zo_done = zo_hi;
        b_done = b_hi;
    }
    if (b_done != n || zo_done != nzo) return api_fail(NRR_E_ARG, "internal: the slab pipeline left %d blocks unmatched", n - b_done);
    NRR_CUDA(cudaMemcpyAsync(out_disp, plan->disp_dev, (size_t)n * 3 * sizeof(int), cudaMemcpyDeviceToHost, s));
    NRR_CUDA(cudaMemcpyAsync(out_ncc, plan->ncc_dev, (size_t)n * sizeof(float), cudaMemcpyDeviceToHost, s));
    return api_check_async(s);
}

int nrr_bm_plan_destroy(nrr_bm_plan *plan)
{
    if (!plan) return NRR_OK;
    if (plan->magic != kPlanMagic) return api_fail(NRR_E_ARG, "not a live nrr_bm_plan");
    cudaDeviceSynchronize();
    if (plan->copy_stream) cudaStreamDestroy(plan->copy_stream);
    plan_free(plan);
    return NRR_OK;
}

int nrr_bm_register_batch(const float *fixed, const float *moving, const int dims[3], const unsigned char *mask,
                          const nrr_bm_setting *settings, int n_settings, int *const *out_blocks, const int *capacity,
                          int *out_n, int *const *out_disp, float *const *out_ncc, void *stream_)
{
    cudaStream_t stream = (cudaStream_t)stream_;
    if (!fixed || !moving || !dims) return api_fail(NRR_E_NULL, "fixed/moving/dims is NULL");
    if (n_settings < 0) return api_fail(NRR_E_ARG, "n_settings = %d < 0", n_settings);
    if (n_settings == 0) return NRR_OK;
    if (!settings || !out_blocks || !capacity || !out_disp || !out_ncc) return api_fail(NRR_E_NULL, "a settings/output array is NULL");
    int rc = NRR_OK;
    for (int a = 0; a < 3; ++a)
        if (dims[a] < 1) return api_fail(NRR_E_DIMS, "dims[%d] = %d < 1", a, dims[a]);
    const Int3 d = i3(dims);
    const size_t nvox = (size_t)d.x * d.y * d.z;
    struct Item { Int3 block, stride, window; double frac; Int3 grid; long long ngrid; int n_cap; };
    std::vector<Item> items((size_t)n_settings);
    for (int s = 0; s < n_settings; ++s) {
        const nrr_bm_setting &st = settings[s];
        if ((rc = api_check_select_args(fixed, dims, st.block, st.stride, st.frac))) return rc;
        if ((rc = check_window(st.window))) return rc;
        if (capacity[s] < 0) return api_fail(NRR_E_ARG, "capacity[%d] = %d < 0", s, capacity[s]);
        if (capacity[s] > 0 && (!out_blocks[s] || !out_disp[s] || !out_ncc[s]))
            return api_fail(NRR_E_NULL, "an output of setting %d is NULL with capacity > 0", s);
        Item &it = items[(size_t)s];
        it.block = i3(st.block); it.stride = i3(st.stride); it.window = i3(st.window); it.frac = st.frac;
        MatchPlan mp;
        if ((rc = match_plan(d, it.block, it.window, moving, fixed, &mp))) return rc;
        it.grid = grid_of(d, it.block, it.stride);
        it.ngrid = (long long)it.grid.x * it.grid.y * it.grid.z;
        if (it.ngrid > 0x7fffffffll) return api_fail(NRR_E_DIMS, "stride grid has %lld positions (limit 2^31-1)", it.ngrid);
        const long long kmax = api_capacity_bound(it.ngrid, it.frac);
        it.n_cap = (int)(kmax < (long long)capacity[s] ? kmax : (long long)capacity[s]);
    }
    unsigned int *err_flag = nullptr;
    if ((rc = api_thread_state(&err_flag, nullptr))) return rc;      // the first CUDA call: every argument was validated above
    typedef std::tuple<int, int, int> T3;
    auto t3 = [](Int3 v) { return T3(v.x, v.y, v.z); };
    // ---- shared work, all on the caller's stream.  Scratch is released in that stream's order, behind the join.
    std::vector<AsyncScratch *> scratch;
    struct Cleanup { std::vector<AsyncScratch *> &v; ~Cleanup() { for (AsyncScratch *a : v) delete a; } } cleanup{scratch};
    auto alloc = [&](size_t bytes, void **out) -> int {
        AsyncScratch *a = new AsyncScratch(stream);
        scratch.push_back(a);
        NRR_CUDA(a->alloc(bytes));
        *out = a->p;
        return NRR_OK;
    };
    // (1) moving-volume normalisers: one volume per distinct block shape
    std::map<T3, float *> inv_sd;
    for (const Item &it : items) {
        if (it.n_cap <= 0 || inv_sd.count(t3(it.block))) continue;
        void *p = nullptr;
        if ((rc = alloc(nvox * sizeof(float), &p))) return rc;
        inv_sd[t3(it.block)] = (float *)p;
        profile_begin(1, stream);
        rc = boxstat_enqueue(moving, d, it.block, (float *)p, stream);
        profile_end(1, stream);
        if (rc) return rc;
    }
    // (2) selections: one variance pass per distinct (block, stride); further fractions reuse its keys.
    //     Settings that share (block, stride, frac) share the block list: the first one selects, the others copy.
    struct Sel { int owner; SelectState *st; };
    std::map<std::tuple<T3, T3, double>, Sel> sels;
    std::map<std::tuple<T3, T3>, void *> key_scratch;
    std::vector<SelectState *> st_of((size_t)n_settings, nullptr);
    std::vector<int> owner_of((size_t)n_settings, -1);
    for (int s = 0; s < n_settings; ++s) {
        const Item &it = items[(size_t)s];
        const auto skey = std::make_tuple(t3(it.block), t3(it.stride), it.frac);
        auto found = sels.find(skey);
        if (found != sels.end() && capacity[found->second.owner] >= it.n_cap) {
            owner_of[(size_t)s] = found->second.owner;
            st_of[(size_t)s] = found->second.st;
            continue;
        }
        const auto kkey = std::make_tuple(t3(it.block), t3(it.stride));
        SelectState *st = nullptr;
        profile_begin(0, stream);
        auto ks = key_scratch.find(kkey);
        if (ks != key_scratch.end() && select_can_share_keys(it.ngrid)) {
            void *p = nullptr;
            if ((rc = alloc(256, &p))) return rc;
            st = (SelectState *)p;
            rc = select_more_enqueue(ks->second, it.block, it.stride, it.grid, it.frac, out_blocks[s], capacity[s], nullptr, st, stream);
        } else {
            void *p = nullptr;
            if ((rc = alloc(select_scratch_bytes(it.ngrid), &p))) return rc;
            rc = select_enqueue(fixed, d, it.block, it.stride, it.grid, it.frac, mask, out_blocks[s], capacity[s], nullptr, p, &st, stream);
            if (ks == key_scratch.end()) key_scratch[kkey] = p;
        }
        profile_end(0, stream);
        if (rc) return rc;
        owner_of[(size_t)s] = s;
        st_of[(size_t)s] = st;
        if (found == sels.end()) sels[skey] = Sel{s, st};
    }
    for (int s = 0; s < n_settings; ++s) {
        const int o = owner_of[(size_t)s];
        if (out_n) NRR_CUDA(cudaMemcpyAsync(out_n + s, &st_of[(size_t)s]->k, sizeof(int), cudaMemcpyDeviceToDevice, stream));
        if (o != s && items[(size_t)s].n_cap > 0)
            NRR_CUDA(cudaMemcpyAsync(out_blocks[s], out_blocks[o], (size_t)items[(size_t)s].n_cap * 3 * sizeof(int), cudaMemcpyDeviceToDevice, stream));
    }
    // (3) fixed-block records: one set per distinct block list and record layout (the layout depends on the block
    //     shape only, not on the window)
    std::map<int, float *> rec_of_owner;
    std::vector<float *> records((size_t)n_settings, nullptr);
    for (int s = 0; s < n_settings; ++s) {
        const Item &it = items[(size_t)s];
        if (it.n_cap <= 0) continue;
        const int o = owner_of[(size_t)s];
        // a sharer's n_cap never exceeds its owner's (it shares only if it fits the owner's capacity)
        const int n_rec = items[(size_t)o].n_cap;
        const size_t bytes = match_records_bytes(it.block, it.window, n_rec);
        if (bytes == 0) continue;                          // this shape's kernel keeps no records
        auto r = rec_of_owner.find(o);
        if (r != rec_of_owner.end()) { records[(size_t)s] = r->second; continue; }
        void *p = nullptr;
        if ((rc = alloc(bytes, &p))) return rc;
        MatchCall c;
        c.fixed = fixed; c.dims = d; c.block = it.block; c.window = it.window; c.blocks = out_blocks[o];
        c.n = n_rec;
        c.n_dev = &st_of[(size_t)s]->k; c.records = (float *)p; c.phase = kMatchPrepOnly; c.err_flag = err_flag; c.stream = stream;
        if ((rc = match_enqueue(c))) return rc;
        rec_of_owner[o] = (float *)p;
        records[(size_t)s] = (float *)p;
    }
    // ---- (4) the matching launches, longest first, round-robin over a few streams that fork from `stream`
    cudaStream_t side[4];
    const int nside = api_side_streams(n_settings < 4 ? n_settings : 4, side);
    if (nside < 1) return api_fail(NRR_E_CUDA, "no side streams");
    cudaEvent_t ev_fork = nullptr;
    NRR_CUDA(cudaEventCreateWithFlags(&ev_fork, cudaEventDisableTiming));
    NRR_CUDA(cudaEventRecord(ev_fork, stream));
    for (int j = 0; j < nside; ++j) NRR_CUDA(cudaStreamWaitEvent(side[j], ev_fork, 0));
    std::vector<int> order((size_t)n_settings);
    for (int s = 0; s < n_settings; ++s) order[(size_t)s] = s;
    auto cost = [&](int s) {
        const Item &it = items[(size_t)s];
        return (double)it.n_cap * it.block.x * it.block.y * it.block.z * (2.0 * it.window.x + 1) * (2.0 * it.window.y + 1) * (2.0 * it.window.z + 1);
    };
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return cost(a) > cost(b); });
    std::vector<double> load((size_t)nside, 0.0);
    for (int s : order) {
        const Item &it = items[(size_t)s];
        if (it.n_cap <= 0) continue;
        int j = 0;
        for (int q = 1; q < nside; ++q) if (load[(size_t)q] < load[(size_t)j]) j = q;
        load[(size_t)j] += cost(s);
        MatchCall c;
        c.fixed = fixed; c.moving = moving; c.inv_sd = inv_sd[t3(it.block)]; c.dims = d; c.block = it.block; c.window = it.window;
        c.blocks = out_blocks[s]; c.n = it.n_cap; c.n_dev = &st_of[(size_t)s]->k; c.out_disp = out_disp[s]; c.out_ncc = out_ncc[s];
        c.err_flag = err_flag; c.stream = side[j];
        if (records[(size_t)s]) { c.records = records[(size_t)s]; c.phase = kMatchKernelOnly; }
        if ((rc = match_enqueue(c))) break;
    }
    // join on every path: the scratch is released in the caller's stream order
    for (int j = 0; j < nside; ++j) {
        cudaEvent_t ev = nullptr;
        if (cudaEventCreateWithFlags(&ev, cudaEventDisableTiming) != cudaSuccess || cudaEventRecord(ev, side[j]) != cudaSuccess ||
            cudaStreamWaitEvent(stream, ev, 0) != cudaSuccess) {
            if (ev) cudaEventDestroy(ev);
            cudaEventDestroy(ev_fork);
            return api_fail(NRR_E_CUDA, "join of a side stream failed");
        }
        cudaEventDestroy(ev);       // released once the recorded work has completed
    }
    cudaEventDestroy(ev_fork);
    return rc;
}

}  // extern "C"
