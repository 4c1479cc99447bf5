// nrr_internal.cuh -- declarations shared by the translation units of libnrr_bm.so (CUDA path only).
// Nothing here is shared with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/nrr_bm.h"

// Kernel launch and dynamic shared memory go through two macros so that the test suite can compile these
// sources as plain C++ against tests/cuda_emul (a fiber-per-thread emulation used by the CPU tests only;
// NRR_EMUL is never defined when the product library is built).
#ifndef NRR_EMUL
#define NRR_LAUNCH(kern, grid, block, smem, stream, ...) (kern)<<<(grid), (block), (smem), (stream)>>>(__VA_ARGS__)
#define NRR_DYN_SMEM(name) extern __shared__ __align__(128) unsigned char name[]
#endif

namespace nrr {

struct Int3 { int x, y, z; };

// ---- error plumbing (nrr_api.cu) --------------------------------------------------------------------
void set_error(const char *fmt, ...);
int cuda_fail(cudaError_t e, const char *what);   // records the message, returns NRR_E_CUDA
void count_launch(int n = 1);
// CUDA-event brackets around a phase on the caller's stream (no-ops unless nrr_bm_profile_enable(1)):
// 0 selection, 1 moving-volume statistics, 2 matching kernel, 3 fixed-block records (prep kernel)
void profile_begin(int phase, cudaStream_t stream);
void profile_end(int phase, cudaStream_t stream);

// helpers of the C boundary shared by nrr_api.cu and nrr_plan.cu
int api_fail(int code, const char *fmt, ...);                       // records the message, returns code
int api_thread_state(unsigned int **err_flag, void **pinned);      // per-thread / per-device state (4 KB pinned buffer)
int api_host_stream(cudaStream_t *s);                              // stream of the *_host entry points
int api_check_async(cudaStream_t s);                               // nrr_bm_check_async_error
int api_check_dims_block(const int dims[3], const int block[3]);
int api_check_select_args(const float *fixed, const int dims[3], const int block[3], const int stride[3], double frac);
long long api_capacity_bound(long long ngrid, double frac);
int api_side_streams(int count, cudaStream_t *out);                // returns how many it provides (<= count)

#define NRR_CUDA(call)                                              \
    do {                                                            \
        cudaError_t e__ = (call);                                   \
        if (e__ != cudaSuccess) return ::nrr::cuda_fail(e__, #call); \
    } while (0)

#define NRR_LAUNCH_CHECK(what)                                        \
    do {                                                              \
        cudaError_t e__ = cudaGetLastError();                         \
        if (e__ != cudaSuccess) return ::nrr::cuda_fail(e__, what);   \
        ::nrr::count_launch();                                        \
    } while (0)

// Per-device caches (function attributes, streams, flags) are indexed by the current device ordinal.
constexpr int kMaxDevices = 64;
inline int current_device()
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) dev = 0;
    return dev;
}

// Library scratch: a private stream-ordered memory pool per device (nrr_api.cu).
cudaError_t scratch_alloc(void **p, size_t bytes, cudaStream_t s);

// Stream-ordered scratch released on scope exit, error paths included.
struct AsyncScratch {
    void *p = nullptr;
    cudaStream_t s;
    explicit AsyncScratch(cudaStream_t st) : s(st) {}
    AsyncScratch(const AsyncScratch &) = delete;
    AsyncScratch &operator=(const AsyncScratch &) = delete;
    ~AsyncScratch() { if (p) cudaFreeAsync(p, s); }
    cudaError_t alloc(size_t bytes) { return scratch_alloc(&p, bytes, s); }
};

// ---- selection (nrr_select.cu) ----------------------------------------------------------------------
// Device-side state of one selection call; lives in library scratch.
struct SelectState {
    unsigned long long prefix;      // radix-select: key bits decided so far
    unsigned long long mask;        // which bits of prefix are decided
    unsigned int n_candidates;      // N: in-mask grid positions
    unsigned int k;                 // K = floor(0.5 + N*frac)
    unsigned int k_remaining;       // still to take inside the current prefix bucket
    unsigned int ticket[8];         // last-CTA-done counters, one per kernel of the sequence
    unsigned int total_selected;    // written by the compaction scan (== K)
    unsigned int undecided;         // connectivity pruning: candidates neither kept nor removed yet
    unsigned int kept;              // connectivity pruning: members of the greedy independent set
};

size_t select_scratch_bytes(long long ngrid);
// connectivity: 0 = none, 6 / 18 / 26 = the paper's face / edge / vertex pattern (reading Q20).
// With a pattern the call polls the device (host_poll: pinned, >= sizeof(SelectState)) between batches of
// pruning rounds, i.e. it synchronises `stream`; selection is pre-operative.
// Enqueues the whole selection sequence. `scratch` must hold select_scratch_bytes(ngrid) bytes.
int select_enqueue(const float *fixed, Int3 dims, Int3 block, Int3 stride, Int3 grid, double frac,
                   const unsigned char *mask, int *out_blocks, int capacity, double *out_var,
                   void *scratch, SelectState **state_out, cudaStream_t stream, int connectivity = 0,
                   SelectState *host_poll = nullptr);

// Another selection on the keys a select_enqueue call left in `scratch` (same image, block, stride, mask; no
// connectivity pattern), for another fraction: K, the digit picks and the compaction only.  `st`: 256 device bytes.
bool select_can_share_keys(long long ngrid);
int select_more_enqueue(void *scratch, Int3 block, Int3 stride, Int3 grid, double frac, int *out_blocks, int capacity,
                        double *out_var, SelectState *st, cudaStream_t stream);

// ---- moving-volume statistics (nrr_boxstat.cu) ------------------------------------------------------
// inv_sd[p] = 1/sqrt(sum over the block with ORIGIN p of (m - mean)^2), 0 for zero-variance blocks,
// for every origin p whose block fits in the volume; other entries are left untouched.
int boxstat_enqueue(const float *moving, Int3 dims, Int3 block, float *inv_sd, cudaStream_t stream);
// The same for the block origins with z in [zo_lo, zo_hi) only (reads the planes zo_lo .. zo_hi + block.z - 2): a caller
// that uploads the volume slab by slab computes the normalisers of each slab as it lands.
int boxstat_enqueue_range(const float *moving, Int3 dims, Int3 block, float *inv_sd, int zo_lo, int zo_hi, cudaStream_t stream);

// ---- matching (nrr_match.cu) ------------------------------------------------------------------------
struct MatchPlan {
    int fast;          // 2: pair kernel (two candidate rows per thread), 1: one row per thread, 0: generic kernel
    int threads;
    int smem_bytes;
    int tma;           // 1: TMA staging
    int candidates;
    int blocks_per_cta;
};
// n: the number of blocks the launch will have (0: unknown / large) -- the pair kernel's grouping depends on it
int match_plan(Int3 dims, Int3 block, Int3 window, const void *moving_ptr, const void *fixed_ptr,
               MatchPlan *plan, int n = 0);

// One matching launch sequence.  The pair kernel works from per-block RECORDS of the fixed image (centred block, pair
// table, 1/sqrt(SS_f): everything that needs only the pre-operative image); a caller that keeps
// them across calls (a plan) passes `records` and enqueues the two phases separately.
enum MatchPhase { kMatchBoth = 0, kMatchPrepOnly = 1, kMatchKernelOnly = 2 };
struct MatchCall {
    const float *fixed = nullptr, *moving = nullptr, *inv_sd = nullptr;
    Int3 dims{}, block{}, window{};
    const int *blocks = nullptr;       // [n][3] centres
    int n = 0;
    // n_dev (nullable, DEVICE): the number of blocks is min(n, *n_dev), read by the kernels themselves, so a caller
    // that only knows an upper bound n on the host (selection still in flight) needs no synchronisation.
    const unsigned int *n_dev = nullptr;
    int *out_disp = nullptr;
    float *out_ncc = nullptr;
    unsigned int *err_flag = nullptr;
    float *records = nullptr;          // match_records_bytes(block, window, n) bytes; NULL with kMatchBoth = call scratch
    MatchPhase phase = kMatchBoth;
    cudaStream_t stream = nullptr;
};
int match_enqueue(const MatchCall &c);
// Bytes of fixed-block records the kernel for this shape wants for n blocks (0: that kernel keeps no records).
size_t match_records_bytes(Int3 block, Int3 window, int n);

// nrr_match_pair.cu: tries the pair kernel; *handled tells whether it took the call.
int match_pair_dispatch(const MatchCall &c, MatchPlan *plan_only, bool *handled);
size_t match_pair_records_bytes(Int3 block, Int3 window, int n);

int match_pair_table(Int3 block, Int3 window, unsigned int *out, int capacity, int info[6]);

// ---- dense-field warp (nrr_warp.cu) -----------------------------------------------------------------
int warp_enqueue(const float *image, Int3 dims, const float *field, float *out, cudaStream_t stream);

// ---- FFMA microbenchmark (nrr_fma_peak.cu) ----------------------------------------------------------
int fp32_peak_measure(double *out_tflops, cudaStream_t stream);
int fp32_microbench(double out[7], cudaStream_t stream);

}  // namespace nrr
