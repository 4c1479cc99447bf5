// nrr_api.cu -- the extern "C" boundary of libnrr_bm.so (include/nrr_bm.h): argument validation, scratch
// management, the host-buffer forms, instrumentation.  Every step of the path itself runs in the kernels of
// nrr_select.cu / nrr_boxstat.cu / nrr_match.cu; nothing here computes on the CPU.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <mutex>
#include <vector>

#include "nrr_internal.cuh"

namespace nrr {

extern float g_tie_band;
extern int g_force_generic;
extern int g_disable_tma;
extern int g_force_rows;
extern int g_pair_g;
extern int g_debug_tx_extra;
extern int g_plan_slabs;
extern int g_boxstat_generic;
extern int g_select_generic;

namespace {

thread_local char t_error[512] = "";
thread_local long long t_launches = 0;
thread_local int t_profile = 0;

struct TimedSpan { int phase; cudaEvent_t e0, e1; };
thread_local std::vector<TimedSpan> *t_spans = nullptr;

// Per-thread, per-device state: a second GPU in the same process gets its own flag, streams and events.
struct DevState {
    unsigned int *err_flag = nullptr;      // device, sticky error bits (kErrBounds | kErrStaging of the kernels)
    cudaStream_t host_stream = nullptr;    // stream of the *_host entry points
    cudaStream_t side_stream = nullptr;    // nrr_bm_register: moving statistics run beside the selection
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    cudaStream_t copy_stream = nullptr;    // nrr_bm_register_host: the intra-operative volume goes up beside the selection
    cudaEvent_t ev_alloc = nullptr, ev_moving = nullptr;
    static constexpr int kSide = 4;
    cudaStream_t side[kSide] = {};         // nrr_bm_register_batch / plans: matching launches spread over streams
};
thread_local DevState t_dev[kMaxDevices];
thread_local void *t_pinned = nullptr;     // small pinned staging buffer (host memory: one per thread)
DevState &ds() { return t_dev[current_device()]; }
#define t_err_flag (ds().err_flag)
#define t_host_stream (ds().host_stream)
#define t_side_stream (ds().side_stream)
#define t_ev_fork (ds().ev_fork)
#define t_ev_join (ds().ev_join)

constexpr size_t kPinnedBytes = 4096;

std::mutex g_pool_mutex;
cudaMemPool_t g_pools[kMaxDevices] = {};

int ensure_thread_state()
{
    if (!t_err_flag) {
        NRR_CUDA(cudaMalloc((void **)&t_err_flag, sizeof(unsigned int)));
        NRR_CUDA(cudaMemset(t_err_flag, 0, sizeof(unsigned int)));
    }
    if (!t_pinned) NRR_CUDA(cudaMallocHost(&t_pinned, kPinnedBytes));
    return NRR_OK;
}

constexpr int kPhases = 4;
thread_local cudaEvent_t t_open[kPhases] = {nullptr, nullptr, nullptr, nullptr};

struct Span {      // brackets a phase with events when profiling is on
    int phase;
    cudaStream_t stream;
    Span(int p, cudaStream_t s) : phase(p), stream(s) { profile_begin(phase, stream); }
    void stop() { profile_end(phase, stream); }
};

int fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(t_error, sizeof(t_error), fmt, ap);
    va_end(ap);
    return code;
}

Int3 i3(const int v[3]) { return Int3{v[0], v[1], v[2]}; }

int check_dims_block(const int dims[3], const int block[3])
{
    if (!dims || !block) return fail(NRR_E_NULL, "dims/block is NULL");
    for (int a = 0; a < 3; ++a) {
        if (dims[a] < 1) return fail(NRR_E_DIMS, "dims[%d] = %d < 1", a, dims[a]);
        if (block[a] < 1 || (block[a] & 1) == 0)
            return fail(NRR_E_BLOCK, "block[%d] = %d must be a positive odd edge length", a, block[a]);
        if (block[a] > dims[a]) return fail(NRR_E_DIMS, "block[%d] = %d exceeds dims[%d] = %d", a, block[a], a, dims[a]);
    }
    return NRR_OK;
}

int check_select_args(const float *fixed, const int dims[3], const int block[3], const int stride[3], double frac,
                      const int *out_blocks, int capacity, const int *out_n)
{
    if (!fixed || !out_n || !stride) return fail(NRR_E_NULL, "fixed/stride/out_n is NULL");
    int rc = check_dims_block(dims, block);
    if (rc) return rc;
    for (int a = 0; a < 3; ++a)
        if (stride[a] < 1) return fail(NRR_E_STRIDE, "stride[%d] = %d < 1", a, stride[a]);
    if (!(frac > 0.0 && frac <= 1.0)) return fail(NRR_E_FRAC, "frac = %g outside (0, 1]", frac);
    if (capacity < 0) return fail(NRR_E_ARG, "capacity = %d < 0", capacity);
    if (capacity > 0 && !out_blocks) return fail(NRR_E_NULL, "out_blocks is NULL with capacity > 0");
    return NRR_OK;
}

int check_match_args(const float *fixed, const float *moving, const int dims[3], const int *blocks, int n,
                     const int block[3], const int window[3], const int *out_disp, const float *out_ncc)
{
    if (!fixed || !moving || !window) return fail(NRR_E_NULL, "fixed/moving/window is NULL");
    int rc = check_dims_block(dims, block);
    if (rc) return rc;
    for (int a = 0; a < 3; ++a)
        if (window[a] < 0) return fail(NRR_E_WINDOW, "window[%d] = %d < 0", a, window[a]);
    if (n < 0) return fail(NRR_E_ARG, "n = %d < 0", n);
    if (n > 0 && (!blocks || !out_disp || !out_ncc)) return fail(NRR_E_NULL, "blocks/out_disp/out_ncc is NULL with n > 0");
    return NRR_OK;
}

Int3 grid_of(const int dims[3], const int block[3], const int stride[3])
{
    Int3 g;
    g.x = (dims[0] - block[0]) / stride[0] + 1;
    g.y = (dims[1] - block[1]) / stride[1] + 1;
    g.z = (dims[2] - block[2]) / stride[2] + 1;
    return g;
}

// Upper bound on K = floor(0.5 + N*frac) over every N <= ngrid.  The device rounds the product and the sum
// separately; a host compiler that contracts them into one FMA can land one lower, hence the + 1.
long long capacity_bound(long long ngrid, double frac)
{
    volatile double prod = (double)ngrid * frac;
    volatile double sum = 0.5 + prod;
    long long k = (long long)floor(sum) + 1;
    if (k > ngrid) k = ngrid;
    if (k < 0) k = 0;
    return k;
}

// Device select; returns K through *out_n after one synchronisation.
int select_device(const float *fixed, const int dims[3], const int block[3], const int stride[3], double frac,
                  const unsigned char *mask, int *out_blocks, int capacity, int *out_n, double *out_var,
                  int *out_ncand, cudaStream_t stream, int connectivity = 0)
{
    int rc = ensure_thread_state();
    if (rc) return rc;
    const Int3 g = grid_of(dims, block, stride);
    const long long ngrid = (long long)g.x * g.y * g.z;
    if (ngrid > 0x7fffffffll) return fail(NRR_E_DIMS, "stride grid has %lld positions (limit 2^31-1)", ngrid);
    AsyncScratch sel_buf(stream);
    NRR_CUDA(sel_buf.alloc(select_scratch_bytes(ngrid)));
    SelectState *st = nullptr;
    Span span(0, stream);
    rc = select_enqueue(fixed, i3(dims), i3(block), i3(stride), g, frac, mask, out_blocks, capacity, out_var, sel_buf.p,
                        &st, stream, connectivity, (SelectState *)((char *)t_pinned + 3072));
    span.stop();
    if (rc) return rc;
    SelectState *h = (SelectState *)t_pinned;
    NRR_CUDA(cudaMemcpyAsync(h, st, sizeof(SelectState), cudaMemcpyDeviceToHost, stream));
    NRR_CUDA(cudaStreamSynchronize(stream));
    *out_n = (int)h->k;
    if (out_ncand) *out_ncand = (int)h->n_candidates;
    if ((int)h->k > capacity)
        return fail(NRR_E_CAPACITY, "K = %u selected blocks exceed capacity = %d", h->k, capacity);
    return NRR_OK;
}

int match_device(const float *fixed, const float *moving, const int dims[3], const int *blocks, int n,
                 const int block[3], const int window[3], int *out_disp, float *out_ncc, cudaStream_t stream)
{
    int rc = ensure_thread_state();
    if (rc) return rc;
    if (n == 0) return NRR_OK;
    MatchPlan plan;
    rc = match_plan(i3(dims), i3(block), i3(window), moving, fixed, &plan);
    if (rc) return rc;
    const size_t nvox = (size_t)dims[0] * dims[1] * dims[2];
    AsyncScratch inv_buf(stream);
    NRR_CUDA(inv_buf.alloc(nvox * sizeof(float)));
    float *inv_sd = (float *)inv_buf.p;
    Span s1(1, stream);
    rc = boxstat_enqueue(moving, i3(dims), i3(block), inv_sd, stream);
    s1.stop();
    if (rc == NRR_OK) {
        MatchCall c;
        c.fixed = fixed; c.moving = moving; c.inv_sd = inv_sd; c.dims = i3(dims); c.block = i3(block); c.window = i3(window);
        c.blocks = blocks; c.n = n; c.out_disp = out_disp; c.out_ncc = out_ncc; c.err_flag = t_err_flag; c.stream = stream;
        rc = match_enqueue(c);
    }
    return rc;
}

// select + match of one pair with no host synchronisation: the matching kernels are launched for an upper bound
// on K known on the host and read K itself from the selection state on the device.
int register_device(const float *fixed, const float *moving, const int dims[3], const int block[3],
                    const int stride[3], const int window[3], double frac, const unsigned char *mask, int *out_blocks,
                    int capacity, int *out_n_dev, int *out_disp, float *out_ncc, cudaStream_t stream,
                    cudaEvent_t moving_ready = nullptr)
{
    // moving_ready (nullable): `moving` is still being written on another stream; only the kernels that read it (the
    // moving statistics, and through the join the matching kernels) wait for the event -- the selection does not.
    int rc = ensure_thread_state();
    if (rc) return rc;
    MatchPlan plan;
    if ((rc = match_plan(i3(dims), i3(block), i3(window), moving, fixed, &plan))) return rc;
    const Int3 g = grid_of(dims, block, stride);
    const long long ngrid = (long long)g.x * g.y * g.z;
    if (ngrid > 0x7fffffffll) return fail(NRR_E_DIMS, "stride grid has %lld positions (limit 2^31-1)", ngrid);
    const long long kmax = capacity_bound(ngrid, frac);
    const int n_cap = (int)(kmax < (long long)capacity ? kmax : (long long)capacity);
    // The moving-volume statistics do not depend on the selection: fork them onto a side stream so that both
    // (each far from filling the GPU for long) overlap; the matching kernels join.
    AsyncScratch inv_buf(stream), sel_buf(stream);      // released in stream order on every path out of here
    float *inv_sd = nullptr;
    bool forked = false;
    if (n_cap > 0) {
        const size_t nvox = (size_t)dims[0] * dims[1] * dims[2];
        NRR_CUDA(inv_buf.alloc(nvox * sizeof(float)));
        inv_sd = (float *)inv_buf.p;
        if (!t_side_stream) {
            NRR_CUDA(cudaStreamCreateWithFlags(&t_side_stream, cudaStreamNonBlocking));
            NRR_CUDA(cudaEventCreateWithFlags(&t_ev_fork, cudaEventDisableTiming));
            NRR_CUDA(cudaEventCreateWithFlags(&t_ev_join, cudaEventDisableTiming));
        }
        NRR_CUDA(cudaEventRecord(t_ev_fork, stream));
        NRR_CUDA(cudaStreamWaitEvent(t_side_stream, t_ev_fork, 0));
        if (moving_ready) NRR_CUDA(cudaStreamWaitEvent(t_side_stream, moving_ready, 0));
        Span s1(1, t_side_stream);
        rc = boxstat_enqueue(moving, i3(dims), i3(block), inv_sd, t_side_stream);
        s1.stop();
        NRR_CUDA(cudaEventRecord(t_ev_join, t_side_stream));
        forked = true;
    }
    // The join (main stream waits for the side stream) is enqueued BEHIND the selection kernels so that the two
    // overlap, and on every path: the scratch buffers are released in the main stream's order.
    auto join = [&]() -> int {
        if (forked && cudaStreamWaitEvent(stream, t_ev_join, 0) != cudaSuccess) return fail(NRR_E_CUDA, "join of the side stream failed");
        return NRR_OK;
    };
    if (rc) { join(); return rc; }
    if (cudaSuccess != sel_buf.alloc(select_scratch_bytes(ngrid))) { join(); return fail(NRR_E_CUDA, "cudaMallocAsync failed"); }
    SelectState *st = nullptr;
    Span span(0, stream);
    rc = select_enqueue(fixed, i3(dims), i3(block), i3(stride), g, frac, mask, out_blocks, capacity, nullptr, sel_buf.p,
                        &st, stream);
    span.stop();
    // The fixed-block records need the selection only: they are made BEFORE the join, beside the moving statistics
    // that still run on the side stream; only the matching kernel waits for both.
    AsyncScratch rec_buf(stream);
    MatchCall c;
    c.fixed = fixed; c.moving = moving; c.inv_sd = inv_sd; c.dims = i3(dims); c.block = i3(block); c.window = i3(window);
    c.blocks = out_blocks; c.n = n_cap; c.n_dev = st ? &st->k : nullptr; c.out_disp = out_disp; c.out_ncc = out_ncc;
    c.err_flag = t_err_flag; c.stream = stream;
    const size_t rec_bytes = n_cap > 0 ? match_records_bytes(c.block, c.window, n_cap) : 0;
    if (rc == NRR_OK && rec_bytes > 0) {
        if (rec_buf.alloc(rec_bytes) != cudaSuccess) rc = fail(NRR_E_CUDA, "cudaMallocAsync of the block records failed");
        else {
            c.records = (float *)rec_buf.p;
            c.phase = kMatchPrepOnly;
            rc = match_enqueue(c);
            c.phase = kMatchKernelOnly;
        }
    }
    const int jrc = join();
    if (rc == NRR_OK) rc = jrc;
    if (rc == NRR_OK && n_cap > 0) rc = match_enqueue(c);
    // K goes out BEHIND the matching kernel: a copy node in front of it would only delay the time-critical launch
    // (the selection state lives in call scratch that is released, in stream order, after this copy)
    if (rc == NRR_OK && out_n_dev)
        rc = cudaMemcpyAsync(out_n_dev, &st->k, sizeof(int), cudaMemcpyDeviceToDevice, stream) == cudaSuccess
                 ? NRR_OK : fail(NRR_E_CUDA, "copy of K failed");
    return rc;
}

int check_async(cudaStream_t stream)
{
    int rc = ensure_thread_state();
    if (rc) return rc;
    unsigned int *h = (unsigned int *)((char *)t_pinned + 1024);
    NRR_CUDA(cudaMemcpyAsync(h, t_err_flag, sizeof(unsigned int), cudaMemcpyDeviceToHost, stream));
    NRR_CUDA(cudaMemsetAsync(t_err_flag, 0, sizeof(unsigned int), stream));
    NRR_CUDA(cudaStreamSynchronize(stream));
    if (*h & 2u) return fail(NRR_E_DEVICE, "a staged copy (TMA / bulk) of a matching kernel did not complete");
    if (*h & 1u) return fail(NRR_E_BOUNDS, "a supplied block leaves the volume");
    return NRR_OK;
}

int host_stream(cudaStream_t *s)
{
    if (!t_host_stream) NRR_CUDA(cudaStreamCreateWithFlags(&t_host_stream, cudaStreamNonBlocking));
    *s = t_host_stream;
    return NRR_OK;
}

struct DevBuf {     // stream-ordered device buffer released on scope exit
    void *p = nullptr;
    cudaStream_t s;
    explicit DevBuf(cudaStream_t st) : s(st) {}
    ~DevBuf() { if (p) cudaFreeAsync(p, s); }
    cudaError_t alloc(size_t bytes) { return scratch_alloc(&p, bytes, s); }
    cudaError_t upload(const void *h, size_t bytes)
    {
        cudaError_t e = alloc(bytes);
        if (e != cudaSuccess) return e;
        return cudaMemcpyAsync(p, h, bytes, cudaMemcpyHostToDevice, s);
    }
};

}  // namespace

// Library scratch comes from a PRIVATE stream-ordered pool per device (the process-wide default pool is left as the
// application configured it); freed scratch stays cached in it, so steady-state calls re-map nothing.
cudaMemPool_t scratch_pool()
{
    const int dev = current_device();
    std::lock_guard<std::mutex> lock(g_pool_mutex);
    if (!g_pools[dev]) {
        cudaMemPoolProps props;
        memset(&props, 0, sizeof(props));
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t pool = nullptr;
        if (cudaMemPoolCreate(&pool, &props) != cudaSuccess) { (void)cudaGetLastError(); return nullptr; }
        unsigned long long keep = ~0ull;
        (void)cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
        g_pools[dev] = pool;
    }
    return g_pools[dev];
}

cudaError_t scratch_alloc(void **p, size_t bytes, cudaStream_t s)
{
    cudaMemPool_t pool = scratch_pool();
    if (!pool) return cudaMallocAsync(p, bytes ? bytes : 1, s);
    return cudaMallocFromPoolAsync(p, bytes ? bytes : 1, pool, s);
}

// ---- helpers shared with nrr_plan.cu
int api_fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(t_error, sizeof(t_error), fmt, ap);
    va_end(ap);
    return code;
}
int api_thread_state(unsigned int **err_flag, void **pinned)
{
    int rc = ensure_thread_state();
    if (rc) return rc;
    if (err_flag) *err_flag = t_err_flag;
    if (pinned) *pinned = t_pinned;
    return NRR_OK;
}
int api_host_stream(cudaStream_t *s) { return host_stream(s); }
int api_check_async(cudaStream_t s) { return check_async(s); }
int api_check_dims_block(const int dims[3], const int block[3]) { return check_dims_block(dims, block); }
int api_check_select_args(const float *fixed, const int dims[3], const int block[3], const int stride[3], double frac)
{
    int dummy = 0;
    return check_select_args(fixed, dims, block, stride, frac, nullptr, 0, &dummy);
}
long long api_capacity_bound(long long ngrid, double frac) { return capacity_bound(ngrid, frac); }
// `count` side streams (created once per thread and device) that fork from / join into a caller's stream
int api_side_streams(int count, cudaStream_t *out)
{
    DevState &d = ds();
    if (count > DevState::kSide) count = DevState::kSide;
    for (int i = 0; i < count; ++i) {
        if (!d.side[i]) NRR_CUDA(cudaStreamCreateWithFlags(&d.side[i], cudaStreamNonBlocking));
        out[i] = d.side[i];
    }
    return count;
}

void set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(t_error, sizeof(t_error), fmt, ap);
    va_end(ap);
}

int cuda_fail(cudaError_t e, const char *what)
{
    snprintf(t_error, sizeof(t_error), "CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), what);
    return NRR_E_CUDA;
}

void count_launch(int n) { t_launches += n; }

void profile_begin(int phase, cudaStream_t stream)
{
    if (!t_profile || phase < 0 || phase >= kPhases || t_open[phase]) return;
    cudaEvent_t e = nullptr;
    if (cudaEventCreate(&e) != cudaSuccess) return;
    cudaEventRecord(e, stream);
    t_open[phase] = e;
}

void profile_end(int phase, cudaStream_t stream)
{
    if (phase < 0 || phase >= kPhases || !t_open[phase]) return;
    cudaEvent_t e1 = nullptr;
    if (cudaEventCreate(&e1) != cudaSuccess) { cudaEventDestroy(t_open[phase]); t_open[phase] = nullptr; return; }
    cudaEventRecord(e1, stream);
    if (!t_spans) t_spans = new std::vector<TimedSpan>();
    t_spans->push_back({phase, t_open[phase], e1});
    t_open[phase] = nullptr;
}

}  // namespace nrr

using namespace nrr;

extern "C" {

int nrr_bm_select_blocks(const float *fixed, const int dims[3], const int block[3], const int stride[3], double frac,
                         const unsigned char *mask, int *out_blocks, int capacity, int *out_n, double *out_var,
                         int *out_ncand, void *stream)
{
    int rc = check_select_args(fixed, dims, block, stride, frac, out_blocks, capacity, out_n);
    if (rc) return rc;
    return select_device(fixed, dims, block, stride, frac, mask, out_blocks, capacity, out_n, out_var, out_ncand,
                         (cudaStream_t)stream);
}

int nrr_bm_select_blocks_pruned(const float *fixed, const int dims[3], const int block[3], const int stride[3],
                                double frac, const unsigned char *mask, int connectivity, int *out_blocks,
                                int capacity, int *out_n, double *out_var, int *out_ncand, void *stream)
{
    int rc = check_select_args(fixed, dims, block, stride, frac, out_blocks, capacity, out_n);
    if (rc) return rc;
    if (connectivity != 0 && connectivity != 6 && connectivity != 18 && connectivity != 26)
        return fail(NRR_E_ARG, "connectivity = %d (0, 6, 18 or 26)", connectivity);
    return select_device(fixed, dims, block, stride, frac, mask, out_blocks, capacity, out_n, out_var, out_ncand,
                         (cudaStream_t)stream, connectivity);
}

int nrr_bm_select_blocks_pruned_host(const float *fixed, const int dims[3], const int block[3], const int stride[3],
                                     double frac, const unsigned char *mask, int connectivity, int *out_blocks,
                                     int capacity, int *out_n, double *out_var, int *out_ncand)
{
    int rc = check_select_args(fixed, dims, block, stride, frac, out_blocks, capacity, out_n);
    if (rc) return rc;
    if (connectivity != 0 && connectivity != 6 && connectivity != 18 && connectivity != 26)
        return fail(NRR_E_ARG, "connectivity = %d (0, 6, 18 or 26)", connectivity);
    if ((rc = ensure_thread_state())) return rc;
    cudaStream_t s;
    if ((rc = host_stream(&s))) return rc;
    const size_t nvox = (size_t)dims[0] * dims[1] * dims[2];
    DevBuf d_fixed(s), d_mask(s), d_blocks(s), d_var(s);
    NRR_CUDA(d_fixed.upload(fixed, nvox * sizeof(float)));
    if (mask) NRR_CUDA(d_mask.upload(mask, nvox));
    NRR_CUDA(d_blocks.alloc((size_t)capacity * 3 * sizeof(int)));
    if (out_var) NRR_CUDA(d_var.alloc((size_t)capacity * sizeof(double)));
    rc = select_device((const float *)d_fixed.p, dims, block, stride, frac, (const unsigned char *)d_mask.p,
                       (int *)d_blocks.p, capacity, out_n, (double *)d_var.p, out_ncand, s, connectivity);
    if (rc != NRR_OK && rc != NRR_E_CAPACITY) return rc;
    const size_t k = (size_t)(*out_n < capacity ? *out_n : capacity);
    NRR_CUDA(cudaMemcpyAsync(out_blocks, d_blocks.p, k * 3 * sizeof(int), cudaMemcpyDeviceToHost, s));
    if (out_var) NRR_CUDA(cudaMemcpyAsync(out_var, d_var.p, k * sizeof(double), cudaMemcpyDeviceToHost, s));
    NRR_CUDA(cudaStreamSynchronize(s));
    return rc;
}

int nrr_bm_match(const float *fixed, const float *moving, const int dims[3], const int *blocks, int n,
                 const int block[3], const int window[3], int *out_disp, float *out_ncc, void *stream)
{
    int rc = check_match_args(fixed, moving, dims, blocks, n, block, window, out_disp, out_ncc);
    if (rc) return rc;
    return match_device(fixed, moving, dims, blocks, n, block, window, out_disp, out_ncc, (cudaStream_t)stream);
}

int nrr_bm_moving_stats(const float *moving, const int dims[3], const int block[3], float *out_inv_sd, void *stream)
{
    if (!moving || !out_inv_sd) return fail(NRR_E_NULL, "moving/out_inv_sd is NULL");
    int rc = check_dims_block(dims, block);
    if (rc) return rc;
    if ((rc = ensure_thread_state())) return rc;
    return boxstat_enqueue(moving, i3(dims), i3(block), out_inv_sd, (cudaStream_t)stream);
}

int nrr_bm_moving_stats_host(const float *moving, const int dims[3], const int block[3], float *out_inv_sd)
{
    if (!moving || !out_inv_sd) return fail(NRR_E_NULL, "moving/out_inv_sd is NULL");
    int rc = check_dims_block(dims, block);
    if (rc) return rc;
    if ((rc = ensure_thread_state())) return rc;
    cudaStream_t s;
    if ((rc = host_stream(&s))) return rc;
    const size_t nvox = (size_t)dims[0] * dims[1] * dims[2];
    DevBuf d_moving(s), d_out(s);
    NRR_CUDA(d_moving.upload(moving, nvox * sizeof(float)));
    NRR_CUDA(d_out.upload(out_inv_sd, nvox * sizeof(float)));      // untouched entries keep the caller's values
    rc = boxstat_enqueue((const float *)d_moving.p, i3(dims), i3(block), (float *)d_out.p, s);
    if (rc) return rc;
    NRR_CUDA(cudaMemcpyAsync(out_inv_sd, d_out.p, nvox * sizeof(float), cudaMemcpyDeviceToHost, s));
    NRR_CUDA(cudaStreamSynchronize(s));
    return NRR_OK;
}

int nrr_bm_register(const float *fixed, const float *moving, const int dims[3], const int block[3], const int stride[3],
                    const int window[3], double frac, const unsigned char *mask, int *out_blocks, int capacity,
                    int *out_n, int *out_disp, float *out_ncc, void *stream)
{
    int dummy = 0;
    int rc = check_select_args(fixed, dims, block, stride, frac, out_blocks, capacity, &dummy);
    if (rc) return rc;
    if (!moving || !window) return fail(NRR_E_NULL, "moving/window is NULL");
    for (int a = 0; a < 3; ++a)
        if (window[a] < 0) return fail(NRR_E_WINDOW, "window[%d] = %d < 0", a, window[a]);
    if (capacity > 0 && (!out_disp || !out_ncc)) return fail(NRR_E_NULL, "out_disp/out_ncc is NULL with capacity > 0");
    return register_device(fixed, moving, dims, block, stride, window, frac, mask, out_blocks, capacity, out_n, out_disp,
                           out_ncc, (cudaStream_t)stream);
}

int nrr_bm_warp(const float *image, const int dims[3], const float *field, float *out, void *stream)
{
    if (!image || !field || !out || !dims) return fail(NRR_E_NULL, "image/dims/field/out is NULL");
    for (int a = 0; a < 3; ++a)
        if (dims[a] < 1) return fail(NRR_E_DIMS, "dims[%d] = %d < 1", a, dims[a]);
    if (image == out) return fail(NRR_E_ARG, "the warp cannot run in place");
    int rc = ensure_thread_state();
    if (rc) return rc;
    return warp_enqueue(image, i3(dims), field, out, (cudaStream_t)stream);
}

int nrr_bm_warp_host(const float *image, const int dims[3], const float *field, float *out)
{
    if (!image || !field || !out || !dims) return fail(NRR_E_NULL, "image/dims/field/out is NULL");
    for (int a = 0; a < 3; ++a)
        if (dims[a] < 1) return fail(NRR_E_DIMS, "dims[%d] = %d < 1", a, dims[a]);
    int rc = ensure_thread_state();
    if (rc) return rc;
    cudaStream_t s;
    if ((rc = host_stream(&s))) return rc;
    const size_t nvox = (size_t)dims[0] * dims[1] * dims[2];
    DevBuf d_img(s), d_field(s), d_out(s);
    NRR_CUDA(d_img.upload(image, nvox * sizeof(float)));
    NRR_CUDA(d_field.upload(field, 3 * nvox * sizeof(float)));
    NRR_CUDA(d_out.alloc(nvox * sizeof(float)));
    rc = warp_enqueue((const float *)d_img.p, i3(dims), (const float *)d_field.p, (float *)d_out.p, s);
    if (rc) return rc;
    NRR_CUDA(cudaMemcpyAsync(out, d_out.p, nvox * sizeof(float), cudaMemcpyDeviceToHost, s));
    NRR_CUDA(cudaStreamSynchronize(s));
    return NRR_OK;
}

int nrr_bm_check_async_error(void *stream) { return check_async((cudaStream_t)stream); }

int nrr_bm_select_blocks_host(const float *fixed, const int dims[3], const int block[3], const int stride[3],
                              double frac, const unsigned char *mask, int *out_blocks, int capacity, int *out_n,
                              double *out_var, int *out_ncand)
{
    int rc = check_select_args(fixed, dims, block, stride, frac, out_blocks, capacity, out_n);
    if (rc) return rc;
    cudaStream_t s;
    if ((rc = host_stream(&s))) return rc;
    const size_t nvox = (size_t)dims[0] * dims[1] * dims[2];
    DevBuf d_fixed(s), d_mask(s), d_blocks(s), d_var(s);
    NRR_CUDA(d_fixed.upload(fixed, nvox * sizeof(float)));
    if (mask) NRR_CUDA(d_mask.upload(mask, nvox));
    NRR_CUDA(d_blocks.alloc((size_t)capacity * 3 * sizeof(int)));
    if (out_var) NRR_CUDA(d_var.alloc((size_t)capacity * sizeof(double)));
    rc = select_device((const float *)d_fixed.p, dims, block, stride, frac, (const unsigned char *)d_mask.p,
                       (int *)d_blocks.p, capacity, out_n, (double *)d_var.p, out_ncand, s);
    if (rc != NRR_OK && rc != NRR_E_CAPACITY) return rc;
    const size_t k = (size_t)(*out_n < capacity ? *out_n : capacity);
    NRR_CUDA(cudaMemcpyAsync(out_blocks, d_blocks.p, k * 3 * sizeof(int), cudaMemcpyDeviceToHost, s));
    if (out_var) NRR_CUDA(cudaMemcpyAsync(out_var, d_var.p, k * sizeof(double), cudaMemcpyDeviceToHost, s));
    NRR_CUDA(cudaStreamSynchronize(s));
    return rc;
}

int nrr_bm_match_host(const float *fixed, const float *moving, const int dims[3], const int *blocks, int n,
                      const int block[3], const int window[3], int *out_disp, float *out_ncc)
{
    int rc = check_match_args(fixed, moving, dims, blocks, n, block, window, out_disp, out_ncc);
    if (rc) return rc;
    if (n == 0) return NRR_OK;
    cudaStream_t s;
    if ((rc = host_stream(&s))) return rc;
    const size_t nvox = (size_t)dims[0] * dims[1] * dims[2];
    DevBuf d_fixed(s), d_moving(s), d_blocks(s), d_disp(s), d_ncc(s);
    NRR_CUDA(d_fixed.upload(fixed, nvox * sizeof(float)));
    NRR_CUDA(d_moving.upload(moving, nvox * sizeof(float)));
    NRR_CUDA(d_blocks.upload(blocks, (size_t)n * 3 * sizeof(int)));
    NRR_CUDA(d_disp.alloc((size_t)n * 3 * sizeof(int)));
    NRR_CUDA(d_ncc.alloc((size_t)n * sizeof(float)));
    rc = match_device((const float *)d_fixed.p, (const float *)d_moving.p, dims, (const int *)d_blocks.p, n, block,
                      window, (int *)d_disp.p, (float *)d_ncc.p, s);
    if (rc) return rc;
    NRR_CUDA(cudaMemcpyAsync(out_disp, d_disp.p, (size_t)n * 3 * sizeof(int), cudaMemcpyDeviceToHost, s));
    NRR_CUDA(cudaMemcpyAsync(out_ncc, d_ncc.p, (size_t)n * sizeof(float), cudaMemcpyDeviceToHost, s));
    return check_async(s);
}

int nrr_bm_register_host(const float *fixed, const float *moving, const int dims[3], const int block[3],
                         const int stride[3], const int window[3], double frac, const unsigned char *mask,
                         int *out_blocks, int capacity, int *out_n, int *out_disp, float *out_ncc)
{
    int rc = check_select_args(fixed, dims, block, stride, frac, out_blocks, capacity, out_n);
    if (rc) return rc;
    if (!moving || !window) return fail(NRR_E_NULL, "moving/window is NULL");
    for (int a = 0; a < 3; ++a)
        if (window[a] < 0) return fail(NRR_E_WINDOW, "window[%d] = %d < 0", a, window[a]);
    if (capacity > 0 && (!out_disp || !out_ncc)) return fail(NRR_E_NULL, "out_disp/out_ncc is NULL with capacity > 0");
    cudaStream_t s;
    if ((rc = host_stream(&s))) return rc;
    const size_t nvox = (size_t)dims[0] * dims[1] * dims[2];
    if ((rc = ensure_thread_state())) return rc;
    DevBuf d_fixed(s), d_moving(s), d_mask(s), d_blocks(s), d_disp(s), d_ncc(s);
    // The pre-operative inputs go up first, on the compute stream: the selection needs nothing else.  The
    // intra-operative volume follows on a copy stream, so that it is in flight while the selection kernels run; only
    // the moving statistics and the matching kernels wait for it.
    NRR_CUDA(d_moving.alloc(nvox * sizeof(float)));
    DevState &d = ds();
    if (!d.copy_stream) {
        NRR_CUDA(cudaStreamCreateWithFlags(&d.copy_stream, cudaStreamNonBlocking));
        NRR_CUDA(cudaEventCreateWithFlags(&d.ev_alloc, cudaEventDisableTiming));
        NRR_CUDA(cudaEventCreateWithFlags(&d.ev_moving, cudaEventDisableTiming));
    }
    NRR_CUDA(cudaEventRecord(d.ev_alloc, s));                       // the allocation is ordered on s
    NRR_CUDA(d_fixed.upload(fixed, nvox * sizeof(float)));
    if (mask) NRR_CUDA(d_mask.upload(mask, nvox));
    NRR_CUDA(cudaStreamWaitEvent(d.copy_stream, d.ev_alloc, 0));
    NRR_CUDA(cudaMemcpyAsync(d_moving.p, moving, nvox * sizeof(float), cudaMemcpyHostToDevice, d.copy_stream));
    NRR_CUDA(cudaEventRecord(d.ev_moving, d.copy_stream));
    NRR_CUDA(d_blocks.alloc((size_t)capacity * 3 * sizeof(int)));
    DevBuf d_n(s);
    NRR_CUDA(d_n.alloc(sizeof(int)));
    NRR_CUDA(d_disp.alloc((size_t)capacity * 3 * sizeof(int)));
    NRR_CUDA(d_ncc.alloc((size_t)capacity * sizeof(float)));
    rc = register_device((const float *)d_fixed.p, (const float *)d_moving.p, dims, block, stride, window, frac,
                         (const unsigned char *)d_mask.p, (int *)d_blocks.p, capacity, (int *)d_n.p, (int *)d_disp.p,
                         (float *)d_ncc.p, s, d.ev_moving);
    // on every path the compute stream is ordered behind the upload before the buffer is released on it
    if (cudaStreamWaitEvent(s, d.ev_moving, 0) != cudaSuccess && rc == NRR_OK) rc = fail(NRR_E_CUDA, "join of the copy stream failed");
    if (rc) return rc;
    int *h_n = (int *)((char *)t_pinned + 2048);
    NRR_CUDA(cudaMemcpyAsync(h_n, d_n.p, sizeof(int), cudaMemcpyDeviceToHost, s));
    NRR_CUDA(cudaStreamSynchronize(s));
    *out_n = *h_n;
    if (*out_n > capacity) return fail(NRR_E_CAPACITY, "K = %d selected blocks exceed capacity = %d", *out_n, capacity);
    const int n = *out_n;
    if (n == 0) return NRR_OK;
    NRR_CUDA(cudaMemcpyAsync(out_blocks, d_blocks.p, (size_t)n * 3 * sizeof(int), cudaMemcpyDeviceToHost, s));
    NRR_CUDA(cudaMemcpyAsync(out_disp, d_disp.p, (size_t)n * 3 * sizeof(int), cudaMemcpyDeviceToHost, s));
    NRR_CUDA(cudaMemcpyAsync(out_ncc, d_ncc.p, (size_t)n * sizeof(float), cudaMemcpyDeviceToHost, s));
    return check_async(s);
}

int nrr_bm_profile_enable(int on)
{
    t_profile = on ? 1 : 0;
    return NRR_OK;
}

int nrr_bm_profile_read(double ms[4], int calls[4])
{
    if (!ms || !calls) return fail(NRR_E_NULL, "ms/calls is NULL");
    for (int i = 0; i < kPhases; ++i) { ms[i] = 0.0; calls[i] = 0; }
    if (!t_spans) return NRR_OK;
    int rc = NRR_OK;
    for (TimedSpan &sp : *t_spans) {
        float t = 0.f;
        cudaError_t e = cudaEventSynchronize(sp.e1);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&t, sp.e0, sp.e1);
        if (e != cudaSuccess) rc = cuda_fail(e, "profile events");
        else if (sp.phase >= 0 && sp.phase < kPhases) { ms[sp.phase] += (double)t; calls[sp.phase] += 1; }
        cudaEventDestroy(sp.e0);
        cudaEventDestroy(sp.e1);
    }
    t_spans->clear();
    return rc;
}

long long nrr_bm_launch_count(int reset)
{
    long long v = t_launches;
    if (reset) t_launches = 0;
    return v;
}

int nrr_bm_match_info(const int dims[3], const int block[3], const int window[3], int info[6])
{
    if (!info || !window) return fail(NRR_E_NULL, "info/window is NULL");
    int rc = check_dims_block(dims, block);
    if (rc) return rc;
    for (int a = 0; a < 3; ++a)
        if (window[a] < 0) return fail(NRR_E_WINDOW, "window[%d] = %d < 0", a, window[a]);
    MatchPlan plan;
    memset(&plan, 0, sizeof(plan));
    rc = match_plan(i3(dims), i3(block), i3(window), nullptr, nullptr, &plan);
    if (rc) return rc;
    info[0] = plan.fast; info[1] = plan.threads; info[2] = plan.smem_bytes; info[3] = plan.tma; info[4] = plan.candidates; info[5] = plan.blocks_per_cta;
    return NRR_OK;
}

int nrr_bm_match_info_n(const int dims[3], const int block[3], const int window[3], int n, int info[6])
{
    if (!info || !window) return fail(NRR_E_NULL, "info/window is NULL");
    int rc = check_dims_block(dims, block);
    if (rc) return rc;
    for (int a = 0; a < 3; ++a)
        if (window[a] < 0) return fail(NRR_E_WINDOW, "window[%d] = %d < 0", a, window[a]);
    if (n < 0) return fail(NRR_E_ARG, "n = %d < 0", n);
    MatchPlan plan;
    memset(&plan, 0, sizeof(plan));
    rc = match_plan(i3(dims), i3(block), i3(window), nullptr, nullptr, &plan, n);
    if (rc) return rc;
    info[0] = plan.fast; info[1] = plan.threads; info[2] = plan.smem_bytes; info[3] = plan.tma; info[4] = plan.candidates; info[5] = plan.blocks_per_cta;
    return NRR_OK;
}

int nrr_bm_pair_task_table(const int block[3], const int window[3], unsigned int *out_table, int capacity, int info[6])
{
    if (!block || !window || !info || (capacity > 0 && !out_table)) return fail(NRR_E_NULL, "block/window/info/out_table is NULL");
    const int n = match_pair_table(i3(block), i3(window), out_table, capacity, info);
    if (n < 0) return fail(NRR_E_CAPACITY, "the table has %d entries, capacity is %d", -n, capacity);
    if (n == 0) return fail(NRR_E_ARG, "the pair kernel has no plan for this block / window");
    return NRR_OK;
}

int nrr_bm_fp32_peak(double *out_tflops, void *stream)
{
    if (!out_tflops) return fail(NRR_E_NULL, "out_tflops is NULL");
    return fp32_peak_measure(out_tflops, (cudaStream_t)stream);
}

int nrr_bm_fp32_microbench(double out_tflops[7], void *stream)
{
    if (!out_tflops) return fail(NRR_E_NULL, "out_tflops is NULL");
    return fp32_microbench(out_tflops, (cudaStream_t)stream);
}

int nrr_bm_set_option(const char *name, double value)
{
    if (!name) return fail(NRR_E_NULL, "name is NULL");
    if (!strcmp(name, "tie_band")) { g_tie_band = (float)value; return NRR_OK; }
    if (!strcmp(name, "force_generic")) { g_force_generic = value != 0.0; return NRR_OK; }
    if (!strcmp(name, "disable_tma")) { g_disable_tma = value != 0.0; return NRR_OK; }
    if (!strcmp(name, "select_generic")) { g_select_generic = value != 0.0; return NRR_OK; }
    if (!strcmp(name, "boxstat_generic")) { g_boxstat_generic = value != 0.0; return NRR_OK; }
    if (!strcmp(name, "force_rows")) { g_force_rows = value != 0.0; return NRR_OK; }
    if (!strcmp(name, "pair_blocks_per_cta")) { g_pair_g = (int)value; return NRR_OK; }
    if (!strcmp(name, "plan_slabs")) { g_plan_slabs = value < 1.0 ? 1 : (int)value; return NRR_OK; }
    if (!strcmp(name, "debug_expect_tx_extra")) { g_debug_tx_extra = (int)value & ~15; return NRR_OK; }
    return fail(NRR_E_ARG, "unknown option '%s'", name);
}

const char *nrr_bm_last_error(void) { return t_error; }

const char *nrr_bm_status_string(int status)
{
    switch (status) {
    case NRR_OK: return "NRR_OK";
    case NRR_E_NULL: return "NRR_E_NULL";
    case NRR_E_DIMS: return "NRR_E_DIMS";
    case NRR_E_BLOCK: return "NRR_E_BLOCK";
    case NRR_E_STRIDE: return "NRR_E_STRIDE";
    case NRR_E_WINDOW: return "NRR_E_WINDOW";
    case NRR_E_FRAC: return "NRR_E_FRAC";
    case NRR_E_CAPACITY: return "NRR_E_CAPACITY";
    case NRR_E_BOUNDS: return "NRR_E_BOUNDS";
    case NRR_E_SMEM: return "NRR_E_SMEM";
    case NRR_E_CUDA: return "NRR_E_CUDA";
    case NRR_E_ARG: return "NRR_E_ARG";
    case NRR_E_DEVICE: return "NRR_E_DEVICE";
    case NRR_E_NOCONV: return "NRR_E_NOCONV";
    default: return "NRR_E_UNKNOWN";
    }
}

int nrr_bm_version(void) { return NRR_BM_VERSION; }

}  // extern "C"
