// nrr_select.cu -- variance-based block selection on the device.
//
//   S1  block statistics : one thread per stride-grid position, two-pass population variance in IEEE
//                          double with explicitly rounded (never contracted) operations, summed in
//                          x-fastest order ("computes the variance within a block").
//   S2  count            : K = floor(0.5 + N*frac) on the device with the same rounded operations
//                          ("0.5 + NFeatures x Fs blocks are selected").
//   S3  top-K            : most-significant-digit radix select over the 64-bit variance keys (6 passes of
//                          11/11/11/11/11/9 bits) -> threshold T and the number of T-valued ties to keep
//                          (lowest candidate index first), then an order-preserving compaction that emits
//                          block centres in ascending candidate index.
//
// No CTA ever waits for another: every multi-CTA step ends with the "last CTA done" ticket pattern, so the
// sequence cannot deadlock whatever the grid size.  All launches go to one stream; the caller synchronises
// once to read K.
#include "nrr_internal.cuh"

namespace nrr {

int g_select_generic = 0;       // != 0: runtime-shaped statistics kernel and the multi-launch radix select

namespace {

constexpr int kRadixBins = 2048;
constexpr int kNumPasses = 6;
__constant__ int c_shift[kNumPasses] = {53, 42, 31, 20, 9, 0};
__constant__ int c_width[kNumPasses] = {11, 11, 11, 11, 11, 9};

constexpr int kStatsThreads = 128;
constexpr int kScanThreads = 256;
constexpr int kItemsPerThread = 8;
constexpr int kChunk = kScanThreads * kItemsPerThread;   // grid positions per CTA in the radix / compaction kernels

// Monotone map variance -> unsigned key. Out-of-mask positions carry var = -1 and map to key 0, below every
// candidate (a candidate's key is >= 1), so they can never be taken while K <= N.
__device__ __forceinline__ unsigned long long key_of(double var)
{
    return var < 0.0 ? 0ull : (unsigned long long)__double_as_longlong(var) + 1ull;
}

__device__ __forceinline__ unsigned int digit_of(unsigned long long key, int pass)
{
    return (unsigned int)(key >> c_shift[pass]) & ((1u << c_width[pass]) - 1u);
}

// Block-wide: the calling CTA (all threads) picks the radix digit of pass `pass` that contains the
// k_remaining-th largest key of the current prefix bucket, from the global histogram `hist`.
__device__ void pick_digit(const unsigned int *hist_, SelectState *st, int pass)
{
    const volatile unsigned int *hist = hist_;      // global (written by other CTAs before the ticket) or shared
    __shared__ unsigned int s_warp[32];
    __shared__ unsigned int s_found_bin, s_found_cum;
    const int nbins = 1 << c_width[pass];
    const int T = blockDim.x;
    const int per = (nbins + T - 1) / T;
    const int tid = threadIdx.x;
    const unsigned int k = st->k_remaining;
    // thread t owns the descending bins  top - t*per - i,  i in [0, per)
    unsigned int local = 0;
    for (int i = 0; i < per; ++i) {
        int bin = nbins - 1 - (tid * per + i);
        if (bin >= 0) local += hist[bin];
    }
    // inclusive scan of `local` over the CTA
    unsigned int incl = local;
    const int lane = tid & 31, warp = tid >> 5;
    for (int o = 1; o < 32; o <<= 1) {
        unsigned int v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
    }
    if (lane == 31) s_warp[warp] = incl;
    if (tid == 0) { s_found_bin = (unsigned int)(nbins - 1); s_found_cum = 0; }
    __syncthreads();
    unsigned int base = 0;
    for (int w = 0; w < warp; ++w) base += s_warp[w];
    incl += base;
    const unsigned int excl = incl - local;
    if (k > 0 && excl < k && k <= incl) {
        unsigned int cum = excl;
        for (int i = 0; i < per; ++i) {
            int bin = nbins - 1 - (tid * per + i);
            if (bin < 0) break;
            unsigned int c = hist[bin];
            if (cum + c >= k) { s_found_bin = (unsigned int)bin; s_found_cum = cum; break; }
            cum += c;
        }
    }
    __syncthreads();
    if (tid == 0) {
        st->prefix |= (unsigned long long)s_found_bin << c_shift[pass];
        st->mask |= (unsigned long long)((1u << c_width[pass]) - 1u) << c_shift[pass];
        st->k_remaining = k - s_found_cum;
    }
}

// Adds the CTA's shared histogram into the global one, then returns true in the last CTA to finish.
__device__ bool flush_hist_and_ticket(unsigned int *s_hist, unsigned int *g_hist, unsigned int *ticket)
{
    __shared__ bool s_last;
    __syncthreads();
    for (int b = threadIdx.x; b < kRadixBins; b += blockDim.x) {
        unsigned int c = s_hist[b];
        if (c) atomicAdd(g_hist + b, c);
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = (atomicAdd(ticket, 1u) == gridDim.x - 1);
    __syncthreads();
    if (s_last) __threadfence();
    return s_last;
}

// Two-pass population variance of the block at origin (ox,oy,oz): every operation individually rounded
// (no contraction), summation in x-fastest order -- the same sequence of IEEE operations as the oracle.
__device__ double block_variance(const float *__restrict__ fixed, Int3 dims, Int3 block, int ox, int oy, int oz)
{
    const double nvox = (double)((long long)block.x * block.y * block.z);
    double s = 0.0;
    for (int z = 0; z < block.z; ++z)
        for (int y = 0; y < block.y; ++y) {
            const float *row = fixed + ((size_t)(oz + z) * dims.y + (oy + y)) * dims.x + ox;
            for (int x = 0; x < block.x; ++x) s = __dadd_rn(s, (double)__ldg(row + x));
        }
    const double mean = __ddiv_rn(s, nvox);
    double q = 0.0;
    for (int z = 0; z < block.z; ++z)
        for (int y = 0; y < block.y; ++y) {
            const float *row = fixed + ((size_t)(oz + z) * dims.y + (oy + y)) * dims.x + ox;
            for (int x = 0; x < block.x; ++x) {
                const double d = __dsub_rn((double)__ldg(row + x), mean);
                q = __dadd_rn(q, __dmul_rn(d, d));
            }
        }
    return __ddiv_rn(q, nvox);
}

// Same arithmetic, same order, for a cubic block of compile-time edge B: the loads of a whole z-plane are
// independent of the running sum, so they are issued ahead of the (inherently serial) chain of additions.
template <int B>
__device__ double block_variance_cubic(const float *__restrict__ fixed, Int3 dims, int ox, int oy, int oz)
{
    constexpr int RY = B <= 7 ? B : (B == 9 ? 5 : 4);      // rows loaded ahead of the additions (<= 49 values)
    // Planes unrolled into one basic block, so that the loads of the next plane are scheduled under the additions of
    // this one (with one plane per trip every plane exposed a full load latency: 14 per block).
    constexpr int ZUNROLL = B <= 7 ? B : 2;
    const double nvox = (double)(B * B * B);
    const size_t plane = (size_t)dims.x * dims.y;
    const float *org = fixed + ((size_t)oz * dims.y + oy) * dims.x + ox;
    double s = 0.0;
#pragma unroll(ZUNROLL)
    for (int z = 0; z < B; ++z) {
#pragma unroll
        for (int y0 = 0; y0 < B; y0 += RY) {
            float v[RY * B];
#pragma unroll
            for (int y = 0; y < RY; ++y)
#pragma unroll
                for (int x = 0; x < B; ++x)
                    if (y0 + y < B) v[y * B + x] = __ldg(org + z * plane + (size_t)(y0 + y) * dims.x + x);
#pragma unroll
            for (int y = 0; y < RY; ++y)
#pragma unroll
                for (int x = 0; x < B; ++x)
                    if (y0 + y < B) s = __dadd_rn(s, (double)v[y * B + x]);
        }
    }
    const double mean = __ddiv_rn(s, nvox);
    double q = 0.0;
#pragma unroll(ZUNROLL)
    for (int z = 0; z < B; ++z) {
#pragma unroll
        for (int y0 = 0; y0 < B; y0 += RY) {
            float v[RY * B];
#pragma unroll
            for (int y = 0; y < RY; ++y)
#pragma unroll
                for (int x = 0; x < B; ++x)
                    if (y0 + y < B) v[y * B + x] = __ldg(org + z * plane + (size_t)(y0 + y) * dims.x + x);
#pragma unroll
            for (int y = 0; y < RY; ++y)
#pragma unroll
                for (int x = 0; x < B; ++x)
                    if (y0 + y < B) {
                        const double d = __dsub_rn((double)v[y * B + x], mean);
                        q = __dadd_rn(q, __dmul_rn(d, d));
                    }
        }
    }
    return __ddiv_rn(q, nvox);
}

// S1 + S2 + radix pass 0.  CB = compile-time cubic block edge, 0 = any block shape.
template <int CB>
__global__ void __launch_bounds__(kStatsThreads)
stats_kernel(const float *__restrict__ fixed, Int3 dims, Int3 block, Int3 stride, Int3 grid, long long ngrid,
             double frac, const unsigned char *__restrict__ mask, double *__restrict__ var,
             unsigned int *hist0, SelectState *st)
{
    __shared__ unsigned int s_hist[kRadixBins];
    for (int b = threadIdx.x; b < kRadixBins; b += kStatsThreads) s_hist[b] = 0;
    __syncthreads();

    const long long g = (long long)blockIdx.x * kStatsThreads + threadIdx.x;
    bool in = false;
    if (g < ngrid) {
        const int i = (int)(g % grid.x);
        const int j = (int)((g / grid.x) % grid.y);
        const int k = (int)(g / ((long long)grid.x * grid.y));
        const int ox = i * stride.x, oy = j * stride.y, oz = k * stride.z;
        const int cx = ox + (block.x - 1) / 2, cy = oy + (block.y - 1) / 2, cz = oz + (block.z - 1) / 2;
        in = (mask == nullptr) || mask[((size_t)cz * dims.y + cy) * dims.x + cx] != 0;
        double v = -1.0;
        if (in) {
            if constexpr (CB > 0) v = block_variance_cubic<CB>(fixed, dims, ox, oy, oz);
            else v = block_variance(fixed, dims, block, ox, oy, oz);
            atomicAdd(&s_hist[digit_of(key_of(v), 0)], 1u);
        }
        var[g] = v;
    }
    const int cnt = __syncthreads_count(in ? 1 : 0);
    if (threadIdx.x == 0 && cnt) atomicAdd(&st->n_candidates, (unsigned int)cnt);

    if (flush_hist_and_ticket(s_hist, hist0, &st->ticket[0])) {
        if (threadIdx.x == 0) {
            const unsigned int n = *((volatile unsigned int *)&st->n_candidates);
            // K = floor(0.5 + N*frac), product and sum rounded separately
            double kd = floor(__dadd_rn(0.5, __dmul_rn((double)n, frac)));
            unsigned int kk = kd <= 0.0 ? 0u : (kd >= (double)n ? n : (unsigned int)kd);
            st->k = kk;
            st->k_remaining = kk;
            st->prefix = 0ull;
            st->mask = 0ull;
        }
        __syncthreads();
        pick_digit(hist0, st, 0);
    }
}

// Radix passes 1..5: histogram of the next digit over the keys that match the decided prefix.
__global__ void __launch_bounds__(kScanThreads)
radix_pass_kernel(const double *__restrict__ var, long long ngrid, unsigned int *hist, SelectState *st, int pass)
{
    __shared__ unsigned int s_hist[kRadixBins];
    for (int b = threadIdx.x; b < kRadixBins; b += kScanThreads) s_hist[b] = 0;
    __syncthreads();
    const unsigned long long prefix = st->prefix, mask = st->mask;
    const long long base = (long long)blockIdx.x * kChunk;
#pragma unroll
    for (int i = 0; i < kItemsPerThread; ++i) {
        const long long g = base + (long long)i * kScanThreads + threadIdx.x;
        if (g < ngrid) {
            const unsigned long long key = key_of(var[g]);
            if ((key & mask) == prefix) atomicAdd(&s_hist[digit_of(key, pass)], 1u);
        }
    }
    if (flush_hist_and_ticket(s_hist, hist, &st->ticket[pass])) pick_digit(hist, st, pass);
}

// Packs (#key > T, #key == T) of a run of grid positions into one 64-bit word so one scan carries both.
__device__ __forceinline__ unsigned long long pack_counts(unsigned int gt, unsigned int eq)
{
    return ((unsigned long long)gt << 32) | eq;
}

__device__ unsigned long long block_exclusive_scan_u64(unsigned long long v, unsigned long long *total)
{
    __shared__ unsigned long long s_w[32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    unsigned long long incl = v;
    for (int o = 1; o < 32; o <<= 1) {
        unsigned long long t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    __syncthreads();   // protect s_w against a previous use
    if (lane == 31) s_w[warp] = incl;
    __syncthreads();
    unsigned long long base = 0, tot = 0;
    for (int w = 0; w < nwarp; ++w) {
        if (w < warp) base += s_w[w];
        tot += s_w[w];
    }
    if (total) *total = tot;
    return base + incl - v;
}

// Per-CTA counts of keys above / equal to the threshold; the last CTA turns them into exclusive offsets.
__global__ void __launch_bounds__(kScanThreads)
count_kernel(const double *__restrict__ var, long long ngrid, unsigned long long *cta_counts,
             unsigned long long *cta_offsets, SelectState *st)
{
    const unsigned long long T = st->prefix;
    const long long base = (long long)blockIdx.x * kChunk + (long long)threadIdx.x * kItemsPerThread;
    unsigned int gt = 0, eq = 0;
#pragma unroll
    for (int i = 0; i < kItemsPerThread; ++i) {
        const long long g = base + i;
        if (g < ngrid) {
            const unsigned long long key = key_of(var[g]);
            gt += key > T;
            eq += key == T;
        }
    }
    unsigned long long tot;
    block_exclusive_scan_u64(pack_counts(gt, eq), &tot);
    __shared__ bool s_last;
    if (threadIdx.x == 0) {
        cta_counts[blockIdx.x] = tot;
        __threadfence();
        s_last = (atomicAdd(&st->ticket[6], 1u) == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    // exclusive scan over all CTA totals, kScanThreads at a time
    __shared__ unsigned long long s_carry;
    if (threadIdx.x == 0) s_carry = 0;
    __syncthreads();
    for (unsigned int start = 0; start < gridDim.x; start += kScanThreads) {
        const unsigned int c = start + threadIdx.x;
        const unsigned long long v = c < gridDim.x ? __ldcg(cta_counts + c) : 0ull;
        unsigned long long t;
        const unsigned long long ex = block_exclusive_scan_u64(v, &t);
        const unsigned long long carry = s_carry;
        if (c < gridDim.x) cta_offsets[c] = carry + ex;
        __syncthreads();
        if (threadIdx.x == 0) s_carry = carry + t;
        __syncthreads();
    }
}

// Order-preserving compaction: position of a kept candidate = #(key > T before it) + min(#(key == T before
// it), ties), and a T-valued candidate is kept iff fewer than `ties` T-valued candidates precede it.
__global__ void __launch_bounds__(kScanThreads)
compact_kernel(const double *__restrict__ var, long long ngrid, Int3 block, Int3 stride, Int3 grid,
               const unsigned long long *__restrict__ cta_offsets, const SelectState *st,
               int *__restrict__ out_blocks, double *__restrict__ out_var, int capacity)
{
    const unsigned int K = st->k;
    if (K == 0) return;
    const unsigned long long T = st->prefix;
    const unsigned int ties = st->k_remaining;
    const long long base = (long long)blockIdx.x * kChunk + (long long)threadIdx.x * kItemsPerThread;
    unsigned long long keys[kItemsPerThread];
    unsigned int gt = 0, eq = 0;
#pragma unroll
    for (int i = 0; i < kItemsPerThread; ++i) {
        const long long g = base + i;
        keys[i] = g < ngrid ? key_of(var[g]) : 0ull;
        gt += keys[i] > T;
        eq += (keys[i] == T) && (g < ngrid);
    }
    const unsigned long long ex = block_exclusive_scan_u64(pack_counts(gt, eq), nullptr) + cta_offsets[blockIdx.x];
    unsigned int gt_before = (unsigned int)(ex >> 32), eq_before = (unsigned int)(ex & 0xffffffffu);
#pragma unroll
    for (int i = 0; i < kItemsPerThread; ++i) {
        const long long g = base + i;
        if (g >= ngrid) break;
        const bool is_gt = keys[i] > T, is_eq = keys[i] == T;
        if (is_gt || (is_eq && eq_before < ties)) {
            const unsigned int pos = gt_before + (eq_before < ties ? eq_before : ties);
            if (pos < (unsigned int)capacity) {
                const int gi = (int)(g % grid.x);
                const int gj = (int)((g / grid.x) % grid.y);
                const int gk = (int)(g / ((long long)grid.x * grid.y));
                out_blocks[3 * (size_t)pos + 0] = gi * stride.x + (block.x - 1) / 2;
                out_blocks[3 * (size_t)pos + 1] = gj * stride.y + (block.y - 1) / 2;
                out_blocks[3 * (size_t)pos + 2] = gk * stride.z + (block.z - 1) / 2;
                if (out_var) out_var[pos] = var[g];
            }
        }
        gt_before += is_gt;
        eq_before += is_eq;
    }
}

// ---- small grids: passes 1..5, the threshold counts and the compaction in ONE single-CTA launch.
// 60,000 keys (config 3) are 59 keys per thread and pass; seven tiny launches cost more than the work.
constexpr int kSmallThreads = 1024;
constexpr int kSmallList = 4096;       // keys (32 KB of shared memory) the single-CTA tail may keep on the side
constexpr long long kSmallLimit = 1ll << 20;      // grid positions up to which the single-CTA tail is used

__global__ void __launch_bounds__(kSmallThreads)
select_small_kernel(const double *__restrict__ var, long long ngrid, Int3 block, Int3 stride, Int3 grid,
                    SelectState *st, int *__restrict__ out_blocks, double *__restrict__ out_var, int capacity,
                    int first_pass)
{
    __shared__ unsigned int s_hist[kRadixBins];
    __shared__ unsigned long long s_carry;
    // Keys that match the prefix decided so far.  A full scan collects them on the side; once they fit, the
    // remaining passes walk this list instead of the whole grid (after two digits the bucket of the K-th key
    // usually holds a few dozen keys).  The histograms, hence the selected set, are the same either way.
    __shared__ unsigned long long s_list[kSmallList];
    __shared__ unsigned int s_nlist;
    const int tid = threadIdx.x;
    bool listed = false;                   // uniform: s_list holds exactly the keys matching (prefix, mask)
    for (int pass = first_pass; pass < kNumPasses; ++pass) {
        for (int b = tid; b < kRadixBins; b += kSmallThreads) s_hist[b] = 0;
        const unsigned int nlist = listed ? s_nlist : 0u;
        __syncthreads();
        const unsigned long long prefix = st->prefix, mask = st->mask;
        if (listed) {
            for (unsigned int i = tid; i < nlist; i += kSmallThreads) {
                const unsigned long long key = s_list[i];
                if ((key & mask) == prefix) atomicAdd(&s_hist[digit_of(key, pass)], 1u);
            }
        } else {
            if (tid == 0) s_nlist = 0u;
            __syncthreads();
            // One CTA cannot hide the latency of one load per thread and trip: kScanAhead independent loads are issued
            // before the first key is used (a full scan of config 3's 60,000 keys is 59 keys per thread).
            constexpr int kScanAhead = 8;
            for (long long g0 = tid; g0 < ngrid; g0 += (long long)kSmallThreads * kScanAhead) {
                double v[kScanAhead];
#pragma unroll
                for (int u = 0; u < kScanAhead; ++u) {
                    const long long g = g0 + (long long)u * kSmallThreads;
                    v[u] = g < ngrid ? var[g] : -1.0;
                }
#pragma unroll
                for (int u = 0; u < kScanAhead; ++u) {
                    if (g0 + (long long)u * kSmallThreads >= ngrid) break;
                    const unsigned long long key = key_of(v[u]);
                    if ((key & mask) == prefix) {
                        atomicAdd(&s_hist[digit_of(key, pass)], 1u);
                        if (mask != 0ull) {        // with no digit decided yet everything matches: not worth listing
                            const unsigned int slot = atomicAdd(&s_nlist, 1u);
                            if (slot < (unsigned int)kSmallList) s_list[slot] = key;
                        }
                    }
                }
            }
        }
        __syncthreads();
        if (!listed && mask != 0ull && s_nlist <= (unsigned int)kSmallList) listed = true;      // same value in every thread
        pick_digit(s_hist, st, pass);      // thread 0 updates *st; the barrier below publishes it to the CTA
        __syncthreads();
    }
    const unsigned int K = st->k;
    if (K == 0) return;
    const unsigned long long T = st->prefix;
    const unsigned int ties = st->k_remaining;
    if (tid == 0) s_carry = 0ull;
    __syncthreads();
    constexpr int IPT = 8;      // consecutive keys per thread and trip: eight independent loads, half the block scans of four
    for (long long start = 0; start < ngrid; start += (long long)kSmallThreads * IPT) {
        const long long base = start + (long long)tid * IPT;
        unsigned long long keys[IPT];
        unsigned int gt = 0, eq = 0;
#pragma unroll
        for (int i = 0; i < IPT; ++i) {
            const long long g = base + i;
            keys[i] = g < ngrid ? key_of(var[g]) : 0ull;
            gt += keys[i] > T;
            eq += (keys[i] == T) && (g < ngrid);
        }
        unsigned long long tot;
        const unsigned long long ex = block_exclusive_scan_u64(pack_counts(gt, eq), &tot) + s_carry;
        unsigned int gt_before = (unsigned int)(ex >> 32), eq_before = (unsigned int)(ex & 0xffffffffu);
#pragma unroll
        for (int i = 0; i < IPT; ++i) {
            const long long g = base + i;
            if (g >= ngrid) break;
            const bool is_gt = keys[i] > T, is_eq = keys[i] == T;
            if (is_gt || (is_eq && eq_before < ties)) {
                const unsigned int pos = gt_before + (eq_before < ties ? eq_before : ties);
                if (pos < (unsigned int)capacity) {
                    const int gi = (int)(g % grid.x);
                    const int gj = (int)((g / grid.x) % grid.y);
                    const int gk = (int)(g / ((long long)grid.x * grid.y));
                    out_blocks[3 * (size_t)pos + 0] = gi * stride.x + (block.x - 1) / 2;
                    out_blocks[3 * (size_t)pos + 1] = gj * stride.y + (block.y - 1) / 2;
                    out_blocks[3 * (size_t)pos + 2] = gk * stride.z + (block.z - 1) / 2;
                    if (out_var) out_var[pos] = var[g];
                }
            }
            gt_before += is_gt;
            eq_before += is_eq;
        }
        __syncthreads();                   // every thread has read s_carry
        if (tid == 0) s_carry += tot;
        __syncthreads();
    }
}

// A further selection on the SAME keys (same image, block, stride, mask) with another fraction: the variances and the
// pass-0 histogram do not depend on the fraction, so only K, the digit picks and the compaction are redone.
__global__ void __launch_bounds__(256)
select_begin_kernel(const unsigned int *hist0, const SelectState *st0, SelectState *st, double frac)
{
    if (threadIdx.x == 0) {
        const unsigned int n = st0->n_candidates;
        double kd = floor(__dadd_rn(0.5, __dmul_rn((double)n, frac)));      // the same rounded operations as stats_kernel
        unsigned int kk = kd <= 0.0 ? 0u : (kd >= (double)n ? n : (unsigned int)kd);
        st->n_candidates = n;
        st->k = kk;
        st->k_remaining = kk;
        st->prefix = 0ull;
        st->mask = 0ull;
    }
    __syncthreads();
    pick_digit(hist0, st, 0);
}

// ---- connectivity pruning (reading Q20): the greedy walk by (variance desc, index asc) that keeps a
// candidate iff no kept candidate is among its pattern neighbours on the candidate grid.  A candidate's fate
// depends only on its HIGHER-priority neighbours, so the walk is the unique fixed point of a local rule that all
// candidates can apply at once, round after round: removed if a higher-priority neighbour is kept, kept if every
// higher-priority neighbour is removed, undecided otherwise.  States only move from undecided to a final value
// and final values are what the rule reads, so in-place, unordered updates reach the same fixed point as the
// sequential walk; the highest-priority undecided candidate always decides, so the rounds terminate.  Taking the
// K highest-priority members of the resulting set (the radix select below) is the walk stopped at K kept.
constexpr unsigned char kUndecided = 0, kKept = 1, kRemoved = 2;
constexpr int kPruneThreads = 256;

__global__ void __launch_bounds__(kPruneThreads)
prune_init_kernel(const double *__restrict__ var, long long ngrid, unsigned char *__restrict__ state, SelectState *st)
{
    const long long g = (long long)blockIdx.x * kPruneThreads + threadIdx.x;
    const bool cand = g < ngrid && var[g] >= 0.0;
    if (g < ngrid) state[g] = cand ? kUndecided : kRemoved;
    const int cnt = __syncthreads_count(cand ? 1 : 0);
    if (threadIdx.x == 0 && cnt) atomicAdd(&st->undecided, (unsigned int)cnt);
}

__global__ void __launch_bounds__(kPruneThreads)
prune_round_kernel(const double *__restrict__ var, long long ngrid, Int3 grid, int reach,
                   unsigned char *state, SelectState *st)
{
    const long long g = (long long)blockIdx.x * kPruneThreads + threadIdx.x;
    int decided = 0, keep = 0;
    if (g < ngrid && ((volatile unsigned char *)state)[g] == kUndecided) {
        const int i = (int)(g % grid.x);
        const int j = (int)((g / grid.x) % grid.y);
        const int k = (int)(g / ((long long)grid.x * grid.y));
        const unsigned long long key = key_of(var[g]);
        bool kept_above = false, undecided_above = false;
        for (int dk = -1; dk <= 1; ++dk)
            for (int dj = -1; dj <= 1; ++dj)
                for (int di = -1; di <= 1; ++di) {
                    const int m = abs(di) + abs(dj) + abs(dk);
                    if (m == 0 || m > reach) continue;
                    const int ni = i + di, nj = j + dj, nk = k + dk;
                    if (ni < 0 || nj < 0 || nk < 0 || ni >= grid.x || nj >= grid.y || nk >= grid.z) continue;
                    const long long n = ((long long)nk * grid.y + nj) * grid.x + ni;
                    const unsigned char s = ((volatile unsigned char *)state)[n];
                    if (s == kRemoved) continue;
                    const unsigned long long nkey = key_of(var[n]);
                    if (!(nkey > key || (nkey == key && n < g))) continue;      // lower priority: irrelevant
                    if (s == kKept) kept_above = true;
                    else undecided_above = true;
                }
        if (kept_above) { state[g] = kRemoved; decided = 1; }
        else if (!undecided_above) { state[g] = kKept; decided = 1; keep = 1; }
    }
    const int nd = __syncthreads_count(decided);
    const int nk = __syncthreads_count(keep);
    if (threadIdx.x == 0) {
        if (nd) atomicSub(&st->undecided, (unsigned int)nd);
        if (nk) atomicAdd(&st->kept, (unsigned int)nk);
    }
}

// Candidates outside the independent set drop out of the ranking (variance -1 = key 0).
__global__ void __launch_bounds__(kPruneThreads)
prune_apply_kernel(double *__restrict__ var, long long ngrid, const unsigned char *__restrict__ state)
{
    const long long g = (long long)blockIdx.x * kPruneThreads + threadIdx.x;
    if (g < ngrid && state[g] != kKept) var[g] = -1.0;
}

// K := min(K, |set|); the radix select starts over on the pruned keys.
__global__ void prune_finish_kernel(SelectState *st)
{
    const unsigned int k = st->k < st->kept ? st->k : st->kept;
    st->k = k;
    st->k_remaining = k;
    st->prefix = 0ull;
    st->mask = 0ull;
    st->ticket[0] = 0u;
}

struct ScratchLayout {
    size_t state, hist, var, counts, offsets, prune, total;
};

ScratchLayout layout(long long ngrid)
{
    ScratchLayout L;
    const size_t nchunks = (size_t)((ngrid + kChunk - 1) / kChunk) + 1;
    size_t off = 0;
    L.state = off;   off += 256;                                            // SelectState (zeroed per call)
    L.hist = off;    off += sizeof(unsigned int) * kRadixBins * kNumPasses; // zeroed per call
    L.var = off;     off += sizeof(double) * (size_t)(ngrid > 0 ? ngrid : 1);
    L.counts = off;  off += sizeof(unsigned long long) * nchunks;
    L.offsets = off; off += sizeof(unsigned long long) * nchunks;
    L.prune = off;   off += ((size_t)(ngrid > 0 ? ngrid : 1) + 15) / 16 * 16;             // one state byte per grid position
    L.total = off;
    return L;
}

}  // namespace

size_t select_scratch_bytes(long long ngrid) { return layout(ngrid).total; }

bool select_can_share_keys(long long ngrid) { return !g_select_generic && ngrid > 0 && ngrid <= kSmallLimit; }

int select_more_enqueue(void *scratch, Int3 block, Int3 stride, Int3 grid, double frac, int *out_blocks, int capacity,
                        double *out_var, SelectState *st, cudaStream_t stream)
{
    const long long ngrid = (long long)grid.x * grid.y * grid.z;
    if (!select_can_share_keys(ngrid)) { set_error("the keys of this grid cannot be shared between selections"); return NRR_E_ARG; }
    const ScratchLayout L = layout(ngrid);
    char *base = (char *)scratch;
    const SelectState *st0 = (const SelectState *)(base + L.state);
    const unsigned int *hist0 = (const unsigned int *)(base + L.hist);
    const double *var = (const double *)(base + L.var);
    NRR_CUDA(cudaMemsetAsync(st, 0, sizeof(SelectState), stream));
    NRR_LAUNCH(select_begin_kernel, 1, 256, 0, stream, hist0, st0, st, frac);
    NRR_LAUNCH_CHECK("select_begin_kernel");
    NRR_LAUNCH(select_small_kernel, 1, kSmallThreads, 0, stream, var, ngrid, block, stride, grid, st, out_blocks, out_var,
               capacity, 1);
    NRR_LAUNCH_CHECK("select_small_kernel");
    return NRR_OK;
}

int select_enqueue(const float *fixed, Int3 dims, Int3 block, Int3 stride, Int3 grid, double frac,
                   const unsigned char *mask, int *out_blocks, int capacity, double *out_var, void *scratch,
                   SelectState **state_out, cudaStream_t stream, int connectivity, SelectState *host_poll)
{
    static_assert(sizeof(SelectState) <= 256, "SelectState must fit its scratch slot");
    const long long ngrid = (long long)grid.x * grid.y * grid.z;
    const ScratchLayout L = layout(ngrid);
    char *base = (char *)scratch;
    SelectState *st = (SelectState *)(base + L.state);
    unsigned int *hist = (unsigned int *)(base + L.hist);
    double *var = (double *)(base + L.var);
    unsigned long long *counts = (unsigned long long *)(base + L.counts);
    unsigned long long *offsets = (unsigned long long *)(base + L.offsets);
    *state_out = st;

    NRR_CUDA(cudaMemsetAsync(base, 0, L.var, stream));   // state + histograms
    if (ngrid == 0) return NRR_OK;

    const unsigned int stats_ctas = (unsigned int)((ngrid + kStatsThreads - 1) / kStatsThreads);
    void (*stats)(const float *, Int3, Int3, Int3, Int3, long long, double, const unsigned char *, double *,
                  unsigned int *, SelectState *) = stats_kernel<0>;
    if (!g_select_generic && block.x == block.y && block.y == block.z) {
        if (block.x == 5) stats = stats_kernel<5>;
        else if (block.x == 7) stats = stats_kernel<7>;
        else if (block.x == 9) stats = stats_kernel<9>;
        else if (block.x == 11) stats = stats_kernel<11>;
    }
    NRR_LAUNCH(stats, stats_ctas, kStatsThreads, 0, stream, fixed, dims, block, stride, grid, ngrid, frac, mask, var,
               hist, st);
    NRR_LAUNCH_CHECK("stats_kernel");
    int first_pass = 1;                 // pass 0 is fused into the statistics kernel
    const unsigned int chunks = (unsigned int)((ngrid + kChunk - 1) / kChunk);
    if (connectivity != 0) {
        if (!host_poll) { set_error("connectivity pruning needs a host polling buffer"); return NRR_E_ARG; }
        const int reach = connectivity == 6 ? 1 : connectivity == 18 ? 2 : 3;
        unsigned char *state = (unsigned char *)(base + L.prune);
        const unsigned int pctas = (unsigned int)((ngrid + kPruneThreads - 1) / kPruneThreads);
        NRR_LAUNCH(prune_init_kernel, pctas, kPruneThreads, 0, stream, var, ngrid, state, st);
        NRR_LAUNCH_CHECK("prune_init_kernel");
        for (long long rounds = 0;; rounds += 8) {
            if (rounds > 4 * ngrid + 64) { set_error("connectivity pruning did not converge"); return NRR_E_CUDA; }
            for (int r = 0; r < 8; ++r) {
                NRR_LAUNCH(prune_round_kernel, pctas, kPruneThreads, 0, stream, var, ngrid, grid, reach, state, st);
                NRR_LAUNCH_CHECK("prune_round_kernel");
            }
            NRR_CUDA(cudaMemcpyAsync(host_poll, st, sizeof(SelectState), cudaMemcpyDeviceToHost, stream));
            NRR_CUDA(cudaStreamSynchronize(stream));
            if (host_poll->undecided == 0) break;
        }
        NRR_LAUNCH(prune_apply_kernel, pctas, kPruneThreads, 0, stream, var, ngrid, state);
        NRR_LAUNCH_CHECK("prune_apply_kernel");
        NRR_LAUNCH(prune_finish_kernel, 1, 1, 0, stream, st);
        NRR_LAUNCH_CHECK("prune_finish_kernel");
        NRR_CUDA(cudaMemsetAsync(hist, 0, sizeof(unsigned int) * kRadixBins, stream));
        first_pass = 0;
    }
    if (!g_select_generic && ngrid <= kSmallLimit) {
        NRR_LAUNCH(select_small_kernel, 1, kSmallThreads, 0, stream, var, ngrid, block, stride, grid, st, out_blocks,
                   out_var, capacity, first_pass);
        NRR_LAUNCH_CHECK("select_small_kernel");
        return NRR_OK;
    }
    for (int pass = first_pass; pass < kNumPasses; ++pass) {
        NRR_LAUNCH(radix_pass_kernel, chunks, kScanThreads, 0, stream, var, ngrid, hist + (size_t)pass * kRadixBins, st, pass);
        NRR_LAUNCH_CHECK("radix_pass_kernel");
    }
    NRR_LAUNCH(count_kernel, chunks, kScanThreads, 0, stream, var, ngrid, counts, offsets, st);
    NRR_LAUNCH_CHECK("count_kernel");
    NRR_LAUNCH(compact_kernel, chunks, kScanThreads, 0, stream, var, ngrid, block, stride, grid, offsets, st, out_blocks,
               out_var, capacity);
    NRR_LAUNCH_CHECK("compact_kernel");
    return NRR_OK;
}

}  // namespace nrr
