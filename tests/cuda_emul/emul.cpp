// TEST INFRASTRUCTURE ONLY -- execution model behind tests/cuda_emul/include/cuda_runtime.h.
//
// A kernel launch runs its CTAs one after another on the calling OS thread.  Inside a CTA every CUDA thread is
// a ucontext fiber; fibers run round-robin and switch only inside the emulated collectives (__syncthreads, warp
// shuffles/votes/reductions, mbarrier waits), so shared-memory atomics are plain operations.  A full pass over
// the fibers without any progress is reported as a deadlock.  TMA copies are performed when a thread first waits on
// their mbarrier (until then the destination holds the 0xFF fill, as an unwaited-for read would see garbage); the
// hardware rules this project measured on B200 are asserted (16-byte aligned inner start coordinate and box
// row, 128-byte aligned shared destination, 16-byte granularity of bulk copies).
#include <stdio.h>
#include <time.h>
#include <ucontext.h>

#include <map>
#include <vector>

#include "include/cuda.h"

#if defined(__SANITIZE_ADDRESS__)      // AddressSanitizer build: tell it about the fiber stacks
#include <sanitizer/common_interface_defs.h>
#define EMUL_ASAN 1
#else
#define EMUL_ASAN 0
#endif

namespace emul {

uint3 g_threadIdx, g_blockIdx;
dim3 g_blockDim, g_gridDim;

namespace {

constexpr size_t kStack = 256 * 1024;

struct Fiber {
    ucontext_t ctx;
    unsigned char *stack = nullptr;      // from the grow-only pool below: launches do not re-allocate (and re-fault) them
    bool done = false;
    uint3 tid;
    int linear, warp, lane;
};

struct WarpState {
    unsigned long long slot[32], result[32];
    unsigned arrived_mask = 0, result_present = 0;
    unsigned gen = 0;
    unsigned live_mask = 0;      // lanes that exist and have not exited
};

// Copies are asynchronous on the hardware: the emulation performs them only when a thread first WAITS on their
// barrier, so a kernel that touches the destination without waiting reads the 0xFF fill, not the data.
struct MBar { long long pending; long long tx_expected, tx_done; unsigned phase; std::vector<std::function<void()>> copies; };

struct Cta {
    std::vector<Fiber> fibers;
    std::vector<WarpState> warps;
    int live = 0;
    int bar_arrived = 0, bar_count_pred = 0, bar_result = 0;
    unsigned bar_gen = 0;
    unsigned long long progress = 0;
    unsigned char *smem_raw = nullptr;
    size_t smem_bytes = 0;
    unsigned char *smem_aligned = nullptr;
    std::map<void *, MBar> mbars;
    const std::function<void()> *body = nullptr;
    ucontext_t sched;
    Fiber *cur = nullptr;
    const void *sched_stack_bottom = nullptr;
    size_t sched_stack_size = 0;
};

Cta *g_cta = nullptr;

// All context switches go through these two, so that the sanitizer (when built with it) follows the stacks.
void switch_to_fiber(Cta *c, Fiber *f)
{
#if EMUL_ASAN
    void *fake = nullptr;
    __sanitizer_start_switch_fiber(&fake, f->stack, kStack);
    swapcontext(&c->sched, &f->ctx);
    __sanitizer_finish_switch_fiber(fake, nullptr, nullptr);
#else
    swapcontext(&c->sched, &f->ctx);
#endif
}
void switch_to_scheduler(Cta *c, Fiber *f, bool final)
{
#if EMUL_ASAN
    void *fake = nullptr;
    __sanitizer_start_switch_fiber(final ? nullptr : &fake, c->sched_stack_bottom, c->sched_stack_size);
    swapcontext(&f->ctx, &c->sched);
    __sanitizer_finish_switch_fiber(fake, nullptr, nullptr);
#else
    (void)final;
    swapcontext(&f->ctx, &c->sched);
#endif
}

void fiber_entry()
{
    Cta *c = g_cta;
#if EMUL_ASAN
    __sanitizer_finish_switch_fiber(nullptr, &c->sched_stack_bottom, &c->sched_stack_size);
#endif
    (*c->body)();
    Fiber *f = c->cur;
    f->done = true;
    c->live--;
    c->warps[f->warp].live_mask &= ~(1u << f->lane);
    c->progress++;
    switch_to_scheduler(c, f, true);
}

void yield()
{
    Cta *c = g_cta;
    Fiber *f = c->cur;
    switch_to_scheduler(c, f, false);
    // resumed: the scheduler has restored cur and the built-in indices
}

// A CTA barrier completes when every live thread has arrived (threads that exited do not count).
void cta_barrier_check(Cta *c)
{
    if (c->bar_arrived > 0 && c->bar_arrived >= c->live) {
        c->bar_result = c->bar_count_pred;
        c->bar_arrived = 0;
        c->bar_count_pred = 0;
        c->bar_gen++;
        c->progress++;
    }
}

void warp_check(WarpState &w)
{
    if (w.arrived_mask && (w.arrived_mask & w.live_mask) == w.live_mask) {
        memcpy(w.result, w.slot, sizeof(w.slot));
        w.result_present = w.arrived_mask;
        w.arrived_mask = 0;
        w.gen++;
        g_cta->progress++;
    }
}

}  // namespace

void trap(const char *why)
{
    fprintf(stderr, "[cuda_emul] fatal: %s (block %u, thread %u)\n", why, g_blockIdx.x, g_threadIdx.x);
    abort();
}

unsigned char *dyn_smem() { return g_cta->smem_aligned; }

void syncthreads() { (void)syncthreads_count(0); }

int syncthreads_count(int pred)
{
    Cta *c = g_cta;
    const unsigned gen = c->bar_gen;
    c->bar_arrived++;
    c->bar_count_pred += pred ? 1 : 0;
    c->progress++;
    cta_barrier_check(c);
    while (c->bar_gen == gen) yield();
    return c->bar_result;
}

void warp_gather(unsigned mask, unsigned long long v, unsigned long long out[32], unsigned *present)
{
    Cta *c = g_cta;
    Fiber *f = c->cur;
    WarpState &w = c->warps[f->warp];
    if (!((mask >> f->lane) & 1)) trap("warp collective called by a lane outside its mask");
    // the kernels of this library only use full-mask collectives: every live lane of the warp must arrive
    const unsigned gen = w.gen;
    w.slot[f->lane] = v;
    w.arrived_mask |= 1u << f->lane;
    c->progress++;
    warp_check(w);
    while (w.gen == gen) yield();
    memcpy(out, w.result, sizeof(w.result));
    *present = w.result_present;
}

void syncwarp(unsigned mask)
{
    unsigned long long out[32];
    unsigned present;
    warp_gather(mask, 0, out, &present);
}

// ---- mbarrier / TMA
void mbar_init(void *bar, unsigned count) { g_cta->mbars[bar] = MBar{(long long)count, 0, 0, 0, {}}; g_cta->progress++; }

static MBar &mbar_of(void *bar)
{
    auto it = g_cta->mbars.find(bar);
    if (it == g_cta->mbars.end()) trap("mbarrier used before mbarrier.init");
    return it->second;
}

void mbar_arrive_expect_tx(void *bar, unsigned bytes)
{
    MBar &m = mbar_of(bar);
    m.tx_expected += bytes;
    m.pending -= 1;
    g_cta->progress++;
}

bool mbar_try_wait(void *bar, unsigned parity)
{
    MBar &m = mbar_of(bar);
    if (parity != 0) trap("the emulation models single-phase mbarriers only");
    if (!m.copies.empty()) {
        for (auto &c : m.copies) c();
        m.copies.clear();
        g_cta->progress++;
    }
    if (m.pending < 0 || m.tx_done > m.tx_expected) trap("mbarrier over-arrived / more bytes than expected");
    if (m.pending == 0 && m.tx_done == m.tx_expected) return true;
    yield();
    return false;
}

void mbar_timeout() { g_cta->progress++; }

void tma_load_3d(void *dst, const void *map_, int x, int y, int z, void *bar)
{
    const CUtensorMap *map = (const CUtensorMap *)map_;
    if (map->rank != 3) trap("tensor map of rank != 3");
    if ((x & 3) != 0) trap("TMA inner start coordinate not a multiple of 16 bytes (faults on B200)");
    if (((uintptr_t)dst & 127) != 0) trap("TMA shared destination not 128-byte aligned");
    const CUtensorMap mp = *map;
    MBar &m = mbar_of(bar);
    m.copies.push_back([mp, dst, x, y, z, &m]() {
        float *d = (float *)dst;
        const long long nx = (long long)mp.dim[0], ny = (long long)mp.dim[1], nz = (long long)mp.dim[2];
        for (unsigned c = 0; c < mp.box[2]; ++c)
            for (unsigned b = 0; b < mp.box[1]; ++b)
                for (unsigned a = 0; a < mp.box[0]; ++a) {
                    const long long gx = (long long)x + a, gy = (long long)y + b, gz = (long long)z + c;
                    float v = 0.f;
                    if (gx >= 0 && gx < nx && gy >= 0 && gy < ny && gz >= 0 && gz < nz)
                        v = *(const float *)((const char *)mp.base + gz * mp.stride_bytes[1] + gy * mp.stride_bytes[0] + gx * 4);
                    *d++ = v;
                }
        m.tx_done += (long long)mp.box[0] * mp.box[1] * mp.box[2] * 4;
    });
    g_cta->progress++;
}

void bulk_load(void *dst, const void *src, unsigned bytes, void *bar)
{
    if ((bytes & 15) || ((uintptr_t)dst & 15) || ((uintptr_t)src & 15)) trap("bulk copy not 16-byte aligned / sized");
    MBar &m = mbar_of(bar);
    m.copies.push_back([dst, src, bytes, &m]() {
        memcpy(dst, src, bytes);
        m.tx_done += bytes;
    });
    g_cta->progress++;
}

// ---- launch
void launch(dim3 grid, dim3 block, size_t smem, const std::function<void()> &body)
{
    const int nthreads = (int)(block.x * block.y * block.z);
    if (nthreads < 1 || nthreads > 1024) trap("bad block size");
    if (smem > 227 * 1024) trap("dynamic shared memory above 227 KB");
    Cta cta;
    cta.body = &body;
    cta.fibers.resize(nthreads);
    cta.warps.resize((nthreads + 31) / 32);
    // The window ends exactly where the allocation ends (a sanitizer build then sees every overrun), and its
    // base promises no more than 16-byte alignment, like the hardware.
    unsigned char *raw = nullptr;
    if (posix_memalign((void **)&raw, 128, 128 + smem + 16) != 0) trap("out of memory");
    cta.smem_raw = raw;
    cta.smem_bytes = 128 + smem + 16;
    cta.smem_aligned = raw + 128 + 16;
    static std::vector<unsigned char *> stack_pool;      // launches are serial: one pool serves them all
    while ((int)stack_pool.size() < nthreads) {
        void *p = nullptr;
        if (posix_memalign(&p, 64, kStack) != 0) trap("out of memory");
        stack_pool.push_back((unsigned char *)p);
    }
    for (int t = 0; t < nthreads; ++t) cta.fibers[t].stack = stack_pool[(size_t)t];
    // scheduling order of the runnable threads inside a CTA (default: ascending thread index)
    int sched_mode = 0;
    unsigned long long rng = 0x9E3779B97F4A7C15ull;
    if (const char *e = getenv("NRR_EMUL_SCHED")) {
        if (!strcmp(e, "reverse")) sched_mode = 1;
        else if (!strncmp(e, "random", 6)) { sched_mode = 2; if (e[6] == ':') rng ^= strtoull(e + 7, nullptr, 10); }
    }
    std::vector<int> order;
    if (sched_mode) {
        order.resize((size_t)nthreads);
        for (int i = 0; i < nthreads; ++i) order[(size_t)i] = sched_mode == 1 ? nthreads - 1 - i : i;
    }
    g_blockDim = block;
    g_gridDim = grid;
    Cta *prev = g_cta;
    g_cta = &cta;
    for (unsigned bz = 0; bz < grid.z; ++bz)
        for (unsigned by = 0; by < grid.y; ++by)
            for (unsigned bx = 0; bx < grid.x; ++bx) {
                g_blockIdx = uint3{bx, by, bz};
                cta.live = nthreads;
                cta.bar_arrived = cta.bar_count_pred = 0;
                cta.mbars.clear();
                // uninitialised shared memory must not look initialised
                memset(cta.smem_raw, 0xFF, cta.smem_bytes);      // NaN as float, -1 as int: a use shows up in the results
                for (WarpState &w : cta.warps) { w.arrived_mask = 0; w.live_mask = 0; }
                for (int t = 0; t < nthreads; ++t) {
                    Fiber &f = cta.fibers[t];
                    f.done = false;
                    f.linear = t;
                    f.warp = t >> 5;
                    f.lane = t & 31;
                    f.tid = uint3{(unsigned)t % block.x, ((unsigned)t / block.x) % block.y, (unsigned)t / (block.x * block.y)};
                    cta.warps[f.warp].live_mask |= 1u << f.lane;
                    getcontext(&f.ctx);
                    f.ctx.uc_stack.ss_sp = f.stack;
                    f.ctx.uc_stack.ss_size = kStack;
                    f.ctx.uc_link = nullptr;
                    makecontext(&f.ctx, (void (*)())fiber_entry, 0);
                }
                int idle_passes = 0;
                while (cta.live > 0) {
                    const unsigned long long before = cta.progress;
                    if (sched_mode == 2) {
                        for (int i = nthreads - 1; i > 0; --i) {
                            rng = rng * 6364136223846793005ull + 1442695040888963407ull;
                            std::swap(order[(size_t)i], order[(size_t)((rng >> 33) % (unsigned long long)(i + 1))]);
                        }
                    }
                    for (int tt = 0; tt < nthreads; ++tt) {
                        // NRR_EMUL_SCHED=reverse|random: another order in which runnable threads take their turns; a
                        // result that depends on it is a missing barrier (a race) in the kernel
                        const int t = order.empty() ? tt : order[(size_t)tt];
                        Fiber &f = cta.fibers[t];
                        if (f.done) continue;
                        cta.cur = &f;
                        g_threadIdx = f.tid;
                        switch_to_fiber(&cta, &f);
                        if (f.done) {      // an exit can complete a barrier / collective the others wait on
                            cta_barrier_check(&cta);
                            warp_check(cta.warps[f.warp]);
                        }
                    }
                    if (cta.progress == before) {
                        if (++idle_passes > 4) trap("deadlock: no thread of the CTA can make progress");
                    } else
                        idle_passes = 0;
                }
            }
    g_cta = prev;
    free(cta.smem_raw);
}

}  // namespace emul

// ------------------------------------------------------------------------------------------ runtime API
static double now_ms()
{
    timespec ts;
    clock_gettime(CLOCK_MONOTONIC, &ts);
    return ts.tv_sec * 1e3 + ts.tv_nsec * 1e-6;
}
cudaError_t cudaGetDevice(int *dev) { *dev = 0; return cudaSuccess; }
cudaError_t cudaDeviceGetAttribute(int *v, cudaDeviceAttr, int) { *v = 148; return cudaSuccess; }
cudaError_t cudaDeviceGetDefaultMemPool(cudaMemPool_t *pool, int) { *pool = nullptr; return cudaSuccess; }
cudaError_t cudaMemPoolSetAttribute(cudaMemPool_t, cudaMemPoolAttr, void *) { return cudaSuccess; }
cudaError_t cudaMalloc(void **p, size_t bytes)
{
    *p = nullptr;
    if (posix_memalign(p, 256, bytes ? bytes : 1) != 0) return cudaErrorEmul;      // exact size: overruns are visible to a sanitizer
    memset(*p, 0xFF, bytes);              // device memory is not zero-initialised: NaN as float, -1 as int
    return cudaSuccess;
}
cudaError_t cudaFree(void *p) { free(p); return cudaSuccess; }
cudaError_t cudaMallocHost(void **p, size_t bytes) { return cudaMalloc(p, bytes); }
cudaError_t cudaMallocAsync(void **p, size_t bytes, cudaStream_t) { return cudaMalloc(p, bytes); }
cudaError_t cudaMemPoolCreate(cudaMemPool_t *pool, const cudaMemPoolProps *) { *pool = (cudaMemPool_t)0x1; return cudaSuccess; }
cudaError_t cudaMallocFromPoolAsync(void **p, size_t bytes, cudaMemPool_t, cudaStream_t) { return cudaMalloc(p, bytes); }
cudaError_t cudaFreeAsync(void *p, cudaStream_t) { free(p); return cudaSuccess; }     // launches are synchronous here
cudaError_t cudaMemset(void *p, int v, size_t bytes) { memset(p, v, bytes); return cudaSuccess; }
cudaError_t cudaMemsetAsync(void *p, int v, size_t bytes, cudaStream_t) { memset(p, v, bytes); return cudaSuccess; }
cudaError_t cudaMemcpyAsync(void *d, const void *s, size_t bytes, cudaMemcpyKind, cudaStream_t) { memcpy(d, s, bytes); return cudaSuccess; }
cudaError_t cudaStreamSynchronize(cudaStream_t) { return cudaSuccess; }
cudaError_t cudaDeviceSynchronize(void) { return cudaSuccess; }
cudaError_t cudaStreamDestroy(cudaStream_t) { return cudaSuccess; }
cudaError_t cudaStreamCreateWithFlags(cudaStream_t *s, unsigned) { *s = nullptr; return cudaSuccess; }
cudaError_t cudaEventCreate(cudaEvent_t *e) { *e = new emulEvent_st{0.0}; return cudaSuccess; }
cudaError_t cudaEventCreateWithFlags(cudaEvent_t *e, unsigned) { return cudaEventCreate(e); }
cudaError_t cudaStreamWaitEvent(cudaStream_t, cudaEvent_t, unsigned) { return cudaSuccess; }     // everything is synchronous here
cudaError_t cudaEventDestroy(cudaEvent_t e) { delete e; return cudaSuccess; }
cudaError_t cudaEventRecord(cudaEvent_t e, cudaStream_t) { e->t_ms = now_ms(); return cudaSuccess; }
cudaError_t cudaEventSynchronize(cudaEvent_t) { return cudaSuccess; }
cudaError_t cudaEventQuery(cudaEvent_t) { return cudaSuccess; }
cudaError_t cudaEventElapsedTime(float *ms, cudaEvent_t a, cudaEvent_t b) { *ms = (float)(b->t_ms - a->t_ms); return cudaSuccess; }
cudaError_t cudaGetLastError(void) { return cudaSuccess; }
const char *cudaGetErrorString(cudaError_t e) { return e == cudaSuccess ? "no error" : "emulation error"; }

static CUresult emulTensorMapEncodeTiled(CUtensorMap *map, CUtensorMapDataType dt, cuuint32_t rank, void *base,
                                         const cuuint64_t *gdim, const cuuint64_t *gstride, const cuuint32_t *box,
                                         const cuuint32_t *estride, CUtensorMapInterleave, CUtensorMapSwizzle,
                                         CUtensorMapL2promotion, CUtensorMapFloatOOBfill)
{
    if (dt != CU_TENSOR_MAP_DATA_TYPE_FLOAT32 || rank != 3) return CUDA_ERROR_INVALID_VALUE;
    if (((uintptr_t)base & 15) != 0) return CUDA_ERROR_INVALID_VALUE;
    memset(map, 0, sizeof(*map));
    map->base = base;
    map->rank = rank;
    for (int i = 0; i < 3; ++i) {
        if (box[i] < 1 || box[i] > 256 || estride[i] != 1) return CUDA_ERROR_INVALID_VALUE;
        map->dim[i] = gdim[i];
        map->box[i] = box[i];
    }
    if ((box[0] * 4) % 16 != 0) return CUDA_ERROR_INVALID_VALUE;
    for (int i = 0; i < 2; ++i) {
        if (gstride[i] % 16 != 0) return CUDA_ERROR_INVALID_VALUE;
        map->stride_bytes[i] = gstride[i];
    }
    return CUDA_SUCCESS;
}
cudaError_t cudaGetDriverEntryPoint(const char *name, void **fn, unsigned long long, cudaDriverEntryPointQueryResult *q)
{
    if (!strcmp(name, "cuTensorMapEncodeTiled")) {
        *fn = (void *)emulTensorMapEncodeTiled;
        if (q) *q = cudaDriverEntryPointSuccess;
        return cudaSuccess;
    }
    *fn = nullptr;
    if (q) *q = cudaDriverEntryPointSymbolNotFound;
    return cudaSuccess;
}
