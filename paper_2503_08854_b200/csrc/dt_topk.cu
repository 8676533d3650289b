// dt_topk.cu -- device top-k over the per-orbit SNR (hot-path step 10; Algorithm 1
// `FindSignificantResults`; ordering rule of DESIGN.md step 11: SNR descending, ties
// by orbit index ascending, over orbits with hits >= min_hits and finite SNR).
//
// 1. keys: order-preserving 64-bit image of the fp64 SNR (0 = excluded);
// 2. radix select, 8 passes x 8 bits from the top: block-local shared-memory histograms merged with
//    integer atomics, a one-warp kernel walks the 256 bins and narrows (prefix, k_remaining) -> the
//    exact key T of the k-th best and the number r of entries equal to T that still fit;
// 3. ordered compaction (block counts -> single-block exclusive scan -> scatter): keys > T, then the
//    first r keys == T in INDEX order (this is what makes ties deterministic);
// 4. bitonic sort of the <= k candidates on the composite (key descending, index ascending):
//    shared-memory kernel for spans <= 2048, global compare-exchange steps above that.
#include <string.h>

#include <algorithm>

#include "dt_common.cuh"

namespace dt {

namespace {

constexpr int kThreads = 256;
constexpr int kItems = 16;                    // keys per thread in the streaming kernels
constexpr int kChunk = kThreads * kItems;     // 4096 keys per block
constexpr int kSortSpan = 2048;               // elements sorted per block in shared memory

__device__ __forceinline__ unsigned long long order_key(double x)
{
    unsigned long long b = (unsigned long long)__double_as_longlong(x);
    return (b & 0x8000000000000000ull) ? ~b : (b | 0x8000000000000000ull);
}

__global__ void k_keys(const double *__restrict__ snr, const int32_t *__restrict__ hits, int64_t n,
                       int32_t min_hits, unsigned long long *__restrict__ keys)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double x = snr[i];
    const bool ok = isfinite(x) && hits[i] >= min_hits && hits[i] >= 0;
    keys[i] = ok ? order_key(x) : 0ull;
}

// state[0] = prefix (high bits decided so far), state[1] = k remaining, state[2] = total valid,
// state[3] = threshold T (final), state[4] = r ties to take, state[5] = number of keys > T
__global__ void k_hist(const unsigned long long *__restrict__ keys, int64_t n, int pass,
                       const unsigned long long *__restrict__ state, unsigned int *__restrict__ hist)
{
    __shared__ unsigned int sh[256];
    sh[threadIdx.x] = 0;
    __syncthreads();
    const int shift = 56 - 8 * pass;
    const unsigned long long prefix = state[0];
    const unsigned long long himask = (pass == 0) ? 0ull : (~0ull << (shift + 8));
    const int64_t base = (int64_t)blockIdx.x * kChunk;
#pragma unroll 4
    for (int it = 0; it < kItems; ++it) {
        const int64_t i = base + (int64_t)it * kThreads + threadIdx.x;
        if (i < n) {
            const unsigned long long key = keys[i];
            if (key != 0ull && (key & himask) == prefix)
                atomicAdd(&sh[(unsigned)(key >> shift) & 255u], 1u);
        }
    }
    __syncthreads();
    const unsigned int v = sh[threadIdx.x];
    if (v) atomicAdd(&hist[threadIdx.x], v);
}

// One block of 256 threads, thread d owns bin d: an inclusive suffix scan of the histogram finds the bin of the
// k-th best key (the largest d with sum_{d' >= d} hist[d'] >= k_remaining) without walking the bins serially.
__global__ void k_pick(int pass, int32_t k, unsigned long long *state, unsigned int *hist)
{
    __shared__ unsigned long long suf[256];
    const int t = threadIdx.x;
    const unsigned long long c = hist[t];
    const unsigned long long st0 = state[0], st1 = state[1], st5 = state[5], st6 = state[6];
    suf[t] = c;
    __syncthreads();
    for (int off = 1; off < 256; off <<= 1) {
        const unsigned long long v = (t + off < 256) ? suf[t + off] : 0ull;
        __syncthreads();
        suf[t] += v;
        __syncthreads();
    }
    const unsigned long long total = suf[0];
    const unsigned long long above = suf[t] - c;          // keys in the bins above mine
    hist[t] = 0;                                            // every path leaves a clean histogram
    const int shift = 56 - 8 * pass;
    const unsigned long long krem = (pass == 0) ? (unsigned long long)k : st1;
    if (pass == 0) {
        if (total <= krem) {                                // fewer valid entries than k: take all of them
            if (t == 0) {
                state[0] = 0;
                state[1] = 0;
                state[2] = total;
                state[3] = 0;                               // T = 0: every valid key is > T
                state[4] = 0;
                state[5] = 0;
                state[6] = 1;                               // done flag
            }
            return;
        }
        if (t == 0) {
            state[2] = total;
            state[6] = 0;
        }
    } else if (st6) {
        return;
    }
    // exactly one bin qualifies (k_remaining >= 1 and the bins of the current prefix hold >= k_remaining keys)
    if (above < krem && above + c >= krem) {
        const unsigned long long prefix = st0 | (((unsigned long long)t) << shift);
        state[0] = prefix;
        state[1] = krem - above;
        state[5] = ((pass == 0) ? 0ull : st5) + above;
        if (pass == 7) {
            state[3] = prefix;
            state[4] = krem - above;
        }
    }
}

__global__ void k_count(const unsigned long long *__restrict__ keys, int64_t n,
                        const unsigned long long *__restrict__ state, unsigned int *__restrict__ counts)
{
    __shared__ unsigned int s_gt, s_eq;
    if (threadIdx.x == 0) s_gt = s_eq = 0;
    __syncthreads();
    const unsigned long long T = state[3];
    const int64_t base = (int64_t)blockIdx.x * kChunk;
    unsigned int gt = 0, eq = 0;
    for (int it = 0; it < kItems; ++it) {
        const int64_t i = base + (int64_t)it * kThreads + threadIdx.x;
        if (i < n) {
            const unsigned long long key = keys[i];
            gt += (key > T);
            eq += (key == T && key != 0ull);
        }
    }
    for (int d = 16; d > 0; d >>= 1) {
        gt += __shfl_xor_sync(0xffffffffu, gt, d);
        eq += __shfl_xor_sync(0xffffffffu, eq, d);
    }
    if ((threadIdx.x & 31) == 0) {
        atomicAdd(&s_gt, gt);
        atomicAdd(&s_eq, eq);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        counts[2 * blockIdx.x] = s_gt;
        counts[2 * blockIdx.x + 1] = s_eq;
    }
}

// exclusive scan of the per-block (gt, eq) counts, in place, by one block
__global__ void k_scan(unsigned int *counts, int nblocks, unsigned long long *state)
{
    __shared__ unsigned long long carry[2];
    __shared__ unsigned int tmp[2][1024];
    if (threadIdx.x == 0) carry[0] = carry[1] = 0;
    __syncthreads();
    for (int b0 = 0; b0 < nblocks; b0 += 1024) {
        const int b = b0 + threadIdx.x;
        unsigned int v0 = (b < nblocks) ? counts[2 * b] : 0, v1 = (b < nblocks) ? counts[2 * b + 1] : 0;
        tmp[0][threadIdx.x] = v0;
        tmp[1][threadIdx.x] = v1;
        __syncthreads();
        for (int d = 1; d < 1024; d <<= 1) {
            unsigned int a0 = 0, a1 = 0;
            if (threadIdx.x >= d) { a0 = tmp[0][threadIdx.x - d]; a1 = tmp[1][threadIdx.x - d]; }
            __syncthreads();
            tmp[0][threadIdx.x] += a0;
            tmp[1][threadIdx.x] += a1;
            __syncthreads();
        }
        if (b < nblocks) {
            // offsets can exceed 32 bits only for > 4e9 candidates; k is int32 so they cannot
            counts[2 * b] = (unsigned int)(carry[0] + tmp[0][threadIdx.x] - v0);
            counts[2 * b + 1] = (unsigned int)(carry[1] + tmp[1][threadIdx.x] - v1);
        }
        __syncthreads();
        if (threadIdx.x == 1023) {
            carry[0] += tmp[0][1023];
            carry[1] += tmp[1][1023];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) state[7] = carry[0];   // total number of keys > T
}

__global__ void k_scatter(const unsigned long long *__restrict__ keys, int64_t n,
                          const unsigned long long *__restrict__ state,
                          const unsigned int *__restrict__ counts,
                          unsigned long long *__restrict__ cand_key, long long *__restrict__ cand_idx,
                          unsigned long long limit)
{
    // ordered within the block: each thread handles kItems CONSECUTIVE keys
    __shared__ unsigned int sc[2][kThreads];
    const unsigned long long T = state[3], r = state[4], total_gt = state[7];
    const int64_t base = (int64_t)blockIdx.x * kChunk + (int64_t)threadIdx.x * kItems;
    unsigned int gt = 0, eq = 0;
    unsigned long long loc[kItems];
#pragma unroll
    for (int it = 0; it < kItems; ++it) {
        const int64_t i = base + it;
        loc[it] = (i < n) ? keys[i] : 0ull;
        gt += (loc[it] > T);
        eq += (loc[it] == T && loc[it] != 0ull);
    }
    sc[0][threadIdx.x] = gt;
    sc[1][threadIdx.x] = eq;
    __syncthreads();
    for (int d = 1; d < kThreads; d <<= 1) {
        unsigned int a0 = 0, a1 = 0;
        if (threadIdx.x >= d) { a0 = sc[0][threadIdx.x - d]; a1 = sc[1][threadIdx.x - d]; }
        __syncthreads();
        sc[0][threadIdx.x] += a0;
        sc[1][threadIdx.x] += a1;
        __syncthreads();
    }
    unsigned long long pg = (unsigned long long)counts[2 * blockIdx.x] + sc[0][threadIdx.x] - gt;
    unsigned long long pe = (unsigned long long)counts[2 * blockIdx.x + 1] + sc[1][threadIdx.x] - eq;
#pragma unroll
    for (int it = 0; it < kItems; ++it) {
        const unsigned long long key = loc[it];
        if (key > T) {
            if (pg < limit) {            // threshold mode writes at most `limit` entries (top-k: no limit)
                cand_key[pg] = key;
                cand_idx[pg] = base + it;
            }
            ++pg;
        } else if (key == T && key != 0ull) {
            if (pe < r) {
                cand_key[total_gt + pe] = key;
                cand_idx[total_gt + pe] = base + it;
            }
            ++pe;
        }
    }
}

__global__ void k_pad(unsigned long long *cand_key, long long *cand_idx, int64_t m, int64_t m_pad)
{
    const int64_t i = m + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < m_pad) {
        cand_key[i] = 0ull;                       // sorts last (descending)
        cand_idx[i] = 0x7fffffffffffffffll;
    }
}

// "a before b" in the final order
__device__ __forceinline__ bool before(unsigned long long ka, long long ia, unsigned long long kb,
                                       long long ib)
{
    return (ka > kb) || (ka == kb && ia < ib);
}

// bitonic network, stages (kk, j) for j < kSortSpan handled inside shared memory
__global__ void k_bitonic_local(unsigned long long *cand_key, long long *cand_idx, int64_t m_pad,
                                int64_t kk_begin, int64_t kk_end_incl)
{
    __shared__ unsigned long long sk[kSortSpan];
    __shared__ long long si[kSortSpan];
    const int64_t base = (int64_t)blockIdx.x * kSortSpan;
    for (int t = threadIdx.x; t < kSortSpan; t += blockDim.x) {
        sk[t] = cand_key[base + t];
        si[t] = cand_idx[base + t];
    }
    __syncthreads();
    for (int64_t kk = kk_begin; kk <= kk_end_incl; kk <<= 1) {
        int64_t j0 = kk >> 1;
        if (j0 >= kSortSpan) j0 = kSortSpan >> 1;
        for (int64_t j = j0; j > 0; j >>= 1) {
            for (int t = threadIdx.x; t < kSortSpan / 2; t += blockDim.x) {
                const int lo = (int)(((t / j) * 2 * j) + (t % j));
                const int hi = lo + (int)j;
                const bool asc = (((base + lo) & kk) == 0);   // "asc" = final order direction
                const bool lo_first = before(sk[lo], si[lo], sk[hi], si[hi]);
                if (lo_first != asc) {
                    const unsigned long long tk = sk[lo]; sk[lo] = sk[hi]; sk[hi] = tk;
                    const long long ti = si[lo]; si[lo] = si[hi]; si[hi] = ti;
                }
            }
            __syncthreads();
        }
    }
    for (int t = threadIdx.x; t < kSortSpan; t += blockDim.x) {
        cand_key[base + t] = sk[t];
        cand_idx[base + t] = si[t];
    }
}

__global__ void k_bitonic_global(unsigned long long *cand_key, long long *cand_idx, int64_t m_pad,
                                 int64_t kk, int64_t j)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= m_pad / 2) return;
    const int64_t lo = ((t / j) * 2 * j) + (t % j);
    const int64_t hi = lo + j;
    const bool asc = ((lo & kk) == 0);
    const unsigned long long ka = cand_key[lo], kb = cand_key[hi];
    const long long ia = cand_idx[lo], ib = cand_idx[hi];
    if (before(ka, ia, kb, ib) != asc) {
        cand_key[lo] = kb; cand_key[hi] = ka;
        cand_idx[lo] = ib; cand_idx[hi] = ia;
    }
}

__global__ void k_emit(const long long *__restrict__ cand_idx, const double *__restrict__ snr, int64_t m,
                       double *__restrict__ out_snr)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < m) out_snr[i] = snr[cand_idx[i]];
}

template <typename T>
cudaError_t ensure(T *&ptr, int64_t &cap, int64_t need)
{
    if (need <= cap && ptr) return cudaSuccess;
    if (ptr) cudaFree(ptr);
    ptr = nullptr;
    cap = 0;
    cudaError_t e = cudaMalloc((void **)&ptr, (size_t)need * sizeof(T));
    if (e == cudaSuccess) cap = need;
    return e;
}

}  // namespace

#define TK_CHECK(x)                      \
    do {                                 \
        cudaError_t e__ = (x);           \
        if (e__ != cudaSuccess) return e__; \
    } while (0)

cudaError_t topk_device(const double *snr, const int32_t *hits, int64_t n, int32_t k, int32_t min_hits,
                        TopkWorkspace &ws, int64_t *index_out_host, double *snr_out_host,
                        int32_t *n_found, cudaStream_t stream)
{
    *n_found = 0;
    if (n <= 0 || k <= 0) return cudaSuccess;
    const int64_t kk64 = (k < n) ? (int64_t)k : n;
    int64_t m_pad = kSortSpan;
    while (m_pad < kk64) m_pad <<= 1;
    const int nblocks = (int)((n + kChunk - 1) / kChunk);

    TK_CHECK(ensure(ws.keys, ws.n_cap, n));
    {
        int64_t cap = ws.cand_cap;
        TK_CHECK(ensure(ws.cand_key, cap, m_pad));
        cap = ws.cand_cap;
        TK_CHECK(ensure(ws.cand_idx, cap, m_pad));
        ws.cand_cap = cap;
    }
    if (!ws.hist) TK_CHECK(cudaMalloc((void **)&ws.hist, 256 * sizeof(unsigned int)));
    if (!ws.state) TK_CHECK(cudaMalloc((void **)&ws.state, 16 * sizeof(unsigned long long)));
    TK_CHECK(ensure(ws.block_counts, ws.blocks_cap, (int64_t)2 * nblocks));

    TK_CHECK(cudaMemsetAsync(ws.hist, 0, 256 * sizeof(unsigned int), stream));
    TK_CHECK(cudaMemsetAsync(ws.state, 0, 16 * sizeof(unsigned long long), stream));
    k_keys<<<(unsigned)((n + 255) / 256), 256, 0, stream>>>(snr, hits, n, min_hits, ws.keys);
    for (int pass = 0; pass < 8; ++pass) {
        k_hist<<<nblocks, kThreads, 0, stream>>>(ws.keys, n, pass, ws.state, ws.hist);
        k_pick<<<1, 256, 0, stream>>>(pass, (int32_t)kk64, ws.state, ws.hist);
    }
    k_count<<<nblocks, kThreads, 0, stream>>>(ws.keys, n, ws.state, ws.block_counts);
    k_scan<<<1, 1024, 0, stream>>>(ws.block_counts, nblocks, ws.state);
    k_scatter<<<nblocks, kThreads, 0, stream>>>(ws.keys, n, ws.state, ws.block_counts, ws.cand_key,
                                                ws.cand_idx, ~0ull);
    TK_CHECK(cudaGetLastError());

    unsigned long long st[8];
    TK_CHECK(cudaMemcpyAsync(st, ws.state, sizeof st, cudaMemcpyDeviceToHost, stream));
    TK_CHECK(cudaStreamSynchronize(stream));
    const int64_t total_valid = (int64_t)st[2];
    const int64_t m = (total_valid < kk64) ? total_valid : kk64;
    if (m <= 0) return cudaSuccess;

    int64_t mp = kSortSpan;
    while (mp < m) mp <<= 1;
    if (mp > m) k_pad<<<(unsigned)((mp - m + 255) / 256), 256, 0, stream>>>(ws.cand_key, ws.cand_idx, m, mp);
    // bitonic sort of mp elements
    k_bitonic_local<<<(unsigned)(mp / kSortSpan), 512, 0, stream>>>(ws.cand_key, ws.cand_idx, mp, 2,
                                                                   kSortSpan);
    for (int64_t kk = (int64_t)kSortSpan * 2; kk <= mp; kk <<= 1) {
        for (int64_t j = kk >> 1; j >= kSortSpan; j >>= 1)
            k_bitonic_global<<<(unsigned)((mp / 2 + 255) / 256), 256, 0, stream>>>(ws.cand_key, ws.cand_idx,
                                                                                  mp, kk, j);
        k_bitonic_local<<<(unsigned)(mp / kSortSpan), 512, 0, stream>>>(ws.cand_key, ws.cand_idx, mp, kk,
                                                                       kk);
    }
    // reuse the key buffer (fp64-sized) for the emitted SNR values
    double *out_snr = reinterpret_cast<double *>(ws.keys);
    k_emit<<<(unsigned)((m + 255) / 256), 256, 0, stream>>>(ws.cand_idx, snr, m, out_snr);
    TK_CHECK(cudaGetLastError());
    TK_CHECK(cudaMemcpyAsync(index_out_host, ws.cand_idx, (size_t)m * sizeof(long long),
                             cudaMemcpyDeviceToHost, stream));
    TK_CHECK(cudaMemcpyAsync(snr_out_host, out_snr, (size_t)m * sizeof(double), cudaMemcpyDeviceToHost,
                             stream));
    TK_CHECK(cudaStreamSynchronize(stream));
    *n_found = (int32_t)m;
    return cudaSuccess;
}

// Threshold mode (Algorithm 1 `FindSignificantResults`; "detections above an SNR of 5",
// PAPER.md:336): the ordered compaction of the top-k with a GIVEN threshold key -- keys >= key(snr_min), i.e.
// keys > key(snr_min) - 1 -- and no ties to resolve; candidates leave in ascending index order.
__global__ void k_set_threshold(unsigned long long *state, unsigned long long T)
{
    state[3] = T;
    state[4] = 0;
}

cudaError_t threshold_device(const double *snr, const int32_t *hits, int64_t n, double snr_min,
                             int32_t min_hits, int64_t max_out, TopkWorkspace &ws, int64_t *index_out_host,
                             double *snr_out_host, int64_t *n_found, cudaStream_t stream)
{
    *n_found = 0;
    if (n <= 0) return cudaSuccess;
    const int nblocks = (int)((n + kChunk - 1) / kChunk);
    const int64_t cap = std::max<int64_t>(1, std::min<int64_t>(max_out, n));
    TK_CHECK(ensure(ws.keys, ws.n_cap, n));
    {
        int64_t c = ws.cand_cap;
        TK_CHECK(ensure(ws.cand_key, c, cap));
        c = ws.cand_cap;
        TK_CHECK(ensure(ws.cand_idx, c, cap));
        ws.cand_cap = c;
    }
    if (!ws.hist) TK_CHECK(cudaMalloc((void **)&ws.hist, 256 * sizeof(unsigned int)));
    if (!ws.state) TK_CHECK(cudaMalloc((void **)&ws.state, 16 * sizeof(unsigned long long)));
    TK_CHECK(ensure(ws.block_counts, ws.blocks_cap, (int64_t)2 * nblocks));
    // order-preserving key of the threshold (host copy of order_key; -0.0 and +0.0 compare equal in IEEE, so
    // a zero threshold takes the smaller key)
    double th = (snr_min == 0.0) ? -0.0 : snr_min;
    unsigned long long b;
    static_assert(sizeof b == sizeof th, "fp64");
    memcpy(&b, &th, sizeof b);
    const unsigned long long key = (b & 0x8000000000000000ull) ? ~b : (b | 0x8000000000000000ull);
    TK_CHECK(cudaMemsetAsync(ws.state, 0, 16 * sizeof(unsigned long long), stream));
    k_keys<<<(unsigned)((n + 255) / 256), 256, 0, stream>>>(snr, hits, n, min_hits, ws.keys);
    k_set_threshold<<<1, 1, 0, stream>>>(ws.state, key - 1ull);
    k_count<<<nblocks, kThreads, 0, stream>>>(ws.keys, n, ws.state, ws.block_counts);
    k_scan<<<1, 1024, 0, stream>>>(ws.block_counts, nblocks, ws.state);
    k_scatter<<<nblocks, kThreads, 0, stream>>>(ws.keys, n, ws.state, ws.block_counts, ws.cand_key, ws.cand_idx,
                                                (unsigned long long)max_out);
    TK_CHECK(cudaGetLastError());
    unsigned long long st[8];
    TK_CHECK(cudaMemcpyAsync(st, ws.state, sizeof st, cudaMemcpyDeviceToHost, stream));
    TK_CHECK(cudaStreamSynchronize(stream));
    const int64_t total = (int64_t)st[7];
    *n_found = total;
    const int64_t m = std::min<int64_t>(total, max_out);
    if (m <= 0) return cudaSuccess;
    double *out_snr = reinterpret_cast<double *>(ws.keys);      // the key buffer is free again
    k_emit<<<(unsigned)((m + 255) / 256), 256, 0, stream>>>(ws.cand_idx, snr, m, out_snr);
    TK_CHECK(cudaGetLastError());
    if (index_out_host)
        TK_CHECK(cudaMemcpyAsync(index_out_host, ws.cand_idx, (size_t)m * sizeof(long long), cudaMemcpyDeviceToHost, stream));
    if (snr_out_host)
        TK_CHECK(cudaMemcpyAsync(snr_out_host, out_snr, (size_t)m * sizeof(double), cudaMemcpyDeviceToHost, stream));
    return cudaStreamSynchronize(stream);
}

// ---- sparse per-orbit partial sums (exposure-sharded search; dtrack.h dt_partials_*) ---------------------------
// The orbits a shard has hits for (cnt > 0), in ascending index order, with their sums: the same ordered
// compaction, on the key (cnt > 0).
__global__ void k_hit_keys(const int32_t *__restrict__ cnt, int64_t n, unsigned long long *__restrict__ keys)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) keys[i] = cnt[i] > 0 ? 1ull : 0ull;
}
__global__ void k_gather_partials(const long long *__restrict__ idx, int64_t m, const double *__restrict__ S,
                                  const double *__restrict__ Wt, const int32_t *__restrict__ cnt,
                                  double *__restrict__ S_out, double *__restrict__ Wt_out, int32_t *__restrict__ cnt_out)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < m) {
        const long long o = idx[i];
        S_out[i] = S[o];
        Wt_out[i] = Wt[o];
        cnt_out[i] = cnt[o];
    }
}
// S[idx[i]] += S_in[i] ...: the indices of one list are distinct, so plain read-modify-writes; lists are added one
// after the other in the caller's order (ascending exposure range), which fixes the summation order.
__global__ void k_add_partials(const long long *__restrict__ idx, int64_t m, int64_t n, const double *__restrict__ S_in,
                               const double *__restrict__ Wt_in, const int32_t *__restrict__ cnt_in,
                               double *__restrict__ S, double *__restrict__ Wt, int32_t *__restrict__ cnt, int *bad)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < m) {
        const long long o = idx[i];
        if (o < 0 || o >= n) { *bad = 1; return; }
        S[o] += S_in[i];
        Wt[o] += Wt_in[i];
        cnt[o] += cnt_in[i];
    }
}
// SNR from the current sums; orbits marked invalid by the last dt_stack (hits < 0) stay invalid.
__global__ void k_refinalize(int64_t n, const double *__restrict__ S, const double *__restrict__ Wt,
                             const int32_t *__restrict__ cnt, double *__restrict__ snr, int32_t *__restrict__ hits)
{
    const int64_t o = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (o < n && hits[o] >= 0) {
        const int32_t c = cnt[o];
        snr[o] = (c > 0) ? S[o] / sqrt(Wt[o]) : 0.0;
        hits[o] = c;
    }
}

cudaError_t partials_sparse_device(const double *S, const double *Wt, const int32_t *cnt, int64_t n, int64_t max_out,
                                   TopkWorkspace &ws, long long *idx_out_dev, double *S_out_dev, double *Wt_out_dev,
                                   int32_t *cnt_out_dev, int64_t *n_found, cudaStream_t stream)
{
    *n_found = 0;
    if (n <= 0) return cudaSuccess;
    const int nblocks = (int)((n + kChunk - 1) / kChunk);
    TK_CHECK(ensure(ws.keys, ws.n_cap, n));
    if (!ws.state) TK_CHECK(cudaMalloc((void **)&ws.state, 16 * sizeof(unsigned long long)));
    TK_CHECK(ensure(ws.block_counts, ws.blocks_cap, (int64_t)2 * nblocks));
    // cand_key is scratch of k_scatter: it needs max_out entries too
    {
        int64_t c = ws.cand_cap;
        TK_CHECK(ensure(ws.cand_key, c, std::max<int64_t>(1, std::min<int64_t>(max_out, n))));
        ws.cand_cap = c;
        // cand_idx is NOT used: the indices go straight to the caller's buffer
    }
    TK_CHECK(cudaMemsetAsync(ws.state, 0, 16 * sizeof(unsigned long long), stream));      // T = 0, no ties
    k_hit_keys<<<(unsigned)((n + 255) / 256), 256, 0, stream>>>(cnt, n, ws.keys);
    k_count<<<nblocks, kThreads, 0, stream>>>(ws.keys, n, ws.state, ws.block_counts);
    k_scan<<<1, 1024, 0, stream>>>(ws.block_counts, nblocks, ws.state);
    k_scatter<<<nblocks, kThreads, 0, stream>>>(ws.keys, n, ws.state, ws.block_counts, ws.cand_key, idx_out_dev,
                                                (unsigned long long)max_out);
    TK_CHECK(cudaGetLastError());
    unsigned long long st[8];
    TK_CHECK(cudaMemcpyAsync(st, ws.state, sizeof st, cudaMemcpyDeviceToHost, stream));
    TK_CHECK(cudaStreamSynchronize(stream));
    *n_found = (int64_t)st[7];
    const int64_t m = std::min<int64_t>(*n_found, max_out);
    if (m > 0)
        k_gather_partials<<<(unsigned)((m + 255) / 256), 256, 0, stream>>>(idx_out_dev, m, S, Wt, cnt, S_out_dev,
                                                                          Wt_out_dev, cnt_out_dev);
    return cudaGetLastError();
}

cudaError_t partials_add_device(const long long *idx, int64_t m, int64_t n, const double *S_in, const double *Wt_in,
                                const int32_t *cnt_in, double *S, double *Wt, int32_t *cnt, int *bad_dev,
                                cudaStream_t stream)
{
    if (m <= 0) return cudaSuccess;
    k_add_partials<<<(unsigned)((m + 255) / 256), 256, 0, stream>>>(idx, m, n, S_in, Wt_in, cnt_in, S, Wt, cnt, bad_dev);
    return cudaGetLastError();
}

cudaError_t refinalize_device(int64_t n, const double *S, const double *Wt, const int32_t *cnt, double *snr,
                              int32_t *hits, cudaStream_t stream)
{
    if (n <= 0) return cudaSuccess;
    k_refinalize<<<(unsigned)((n + 255) / 256), 256, 0, stream>>>(n, S, Wt, cnt, snr, hits);
    return cudaGetLastError();
}

// ---- threshold mode without any allocation (dtrack.h dt_threshold_noalloc) -------------------------------------
// For callers that must not call cudaMalloc (CUDA graph capture, tight serving loops): the same ordered
// compaction as threshold_device -- same kernels, same order -- over the caller's DEVICE arrays, with every
// intermediate in ONE file-scope device array and every result written to the caller's DEVICE arrays, so the
// call enqueues kernels (and one 8-byte device-to-device copy) and nothing else: no allocation, no host copy, no
// synchronisation.  The array is part of the library image: every GPU that loads the library holds its
// kNoAllocBytes until the process exits.  Its name is a HOST-side stand-in in host code: the address the kernels
// get is the one cudaGetSymbolAddress returns, taken once per device with that device current.  All calls on a
// device share the array, and it keeps the last call's contents: the state words are cleared by every call, the
// key / candidate / block-count regions are fully rewritten before they are read.  Two calls that overlap on
// the GPU (different streams, no ordering between them) race on it.
constexpr int64_t kNoAllocMaxOrbits = 1 << 20;                                         // DT_NOALLOC_MAX_ORBITS
constexpr int64_t kNoAllocBlocks = (kNoAllocMaxOrbits + kChunk - 1) / kChunk;
constexpr size_t kNoAllocKeys = 0;                                                     // [max] u64 keys
constexpr size_t kNoAllocCand = kNoAllocKeys + (size_t)kNoAllocMaxOrbits * 8;          // [max] u64 candidate keys
constexpr size_t kNoAllocCounts = kNoAllocCand + (size_t)kNoAllocMaxOrbits * 8;        // [2 blocks] u32
constexpr size_t kNoAllocState = kNoAllocCounts + ((size_t)kNoAllocBlocks * 8 + 255) / 256 * 256;   // [16] u64
constexpr size_t kNoAllocBytes = kNoAllocState + 256;                                  // 16.0 MiB + 2.25 KiB
static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocBytes];

namespace {

// the first min(total, max_out) candidates' SNR, `total` read on the device (state[7], written by k_scan)
__global__ void k_emit_counted(const long long *__restrict__ cand_idx, const double *__restrict__ snr,
                               const unsigned long long *__restrict__ state, int64_t max_out,
                               double *__restrict__ out_snr)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t m = min((int64_t)state[7], max_out);
    if (i < m) out_snr[i] = snr[cand_idx[i]];
}

constexpr int kNoAllocMaxDevices = 64;
unsigned char *g_noalloc_addr[kNoAllocMaxDevices];      // device address of g_noalloc_scratch, per device ordinal

}  // namespace

int64_t threshold_noalloc_max() { return kNoAllocMaxOrbits; }

// The current device's address of the scratch array (set-up: once per device, that device current).
static cudaError_t noalloc_scratch_address(unsigned char **out)
{
    int dev = -1;
    TK_CHECK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kNoAllocMaxDevices) return cudaErrorInvalidDevice;
    unsigned char *p = __atomic_load_n(&g_noalloc_addr[dev], __ATOMIC_ACQUIRE);
    if (!p) {
        void *sym = nullptr;
        TK_CHECK(cudaGetSymbolAddress(&sym, g_noalloc_scratch));     // the host-side name is NOT this address
        if (!sym) return cudaErrorInvalidSymbol;
        p = static_cast<unsigned char *>(sym);
        __atomic_store_n(&g_noalloc_addr[dev], p, __ATOMIC_RELEASE);   // racing threads store the same value
    }
    *out = p;
    return cudaSuccess;
}

cudaError_t threshold_noalloc_device(const double *snr, const int32_t *hits, int64_t n, double snr_min,
                                     int32_t min_hits, int64_t max_out, long long *index_out_dev,
                                     double *snr_out_dev, long long *n_found_dev, cudaStream_t stream)
{
    if (n < 0 || n > kNoAllocMaxOrbits) return cudaErrorInvalidValue;      // the caller reports the limit
    unsigned char *base = nullptr;
    TK_CHECK(noalloc_scratch_address(&base));
    unsigned long long *keys = reinterpret_cast<unsigned long long *>(base + kNoAllocKeys);
    unsigned long long *cand_key = reinterpret_cast<unsigned long long *>(base + kNoAllocCand);
    unsigned int *counts = reinterpret_cast<unsigned int *>(base + kNoAllocCounts);
    unsigned long long *state = reinterpret_cast<unsigned long long *>(base + kNoAllocState);
    TK_CHECK(cudaMemsetAsync(state, 0, 16 * sizeof(unsigned long long), stream));   // also the count of an empty call
    if (n > 0) {
        const int nblocks = (int)((n + kChunk - 1) / kChunk);
        double th = (snr_min == 0.0) ? -0.0 : snr_min;                     // as threshold_device
        unsigned long long b;
        memcpy(&b, &th, sizeof b);
        const unsigned long long key = (b & 0x8000000000000000ull) ? ~b : (b | 0x8000000000000000ull);
        k_keys<<<(unsigned)((n + 255) / 256), 256, 0, stream>>>(snr, hits, n, min_hits, keys);
        k_set_threshold<<<1, 1, 0, stream>>>(state, key - 1ull);
        k_count<<<nblocks, kThreads, 0, stream>>>(keys, n, state, counts);
        k_scan<<<1, 1024, 0, stream>>>(counts, nblocks, state);
        // at most min(max_out, n) <= kNoAllocMaxOrbits candidates are written
        k_scatter<<<nblocks, kThreads, 0, stream>>>(keys, n, state, counts, cand_key, index_out_dev,
                                                    (unsigned long long)max_out);
        const int64_t cap = std::min<int64_t>(max_out, n);
        if (snr_out_dev && cap > 0)
            k_emit_counted<<<(unsigned)((cap + 255) / 256), 256, 0, stream>>>(index_out_dev, snr, state, max_out,
                                                                             snr_out_dev);
        TK_CHECK(cudaGetLastError());
    }
    return cudaMemcpyAsync(n_found_dev, state + 7, sizeof(long long), cudaMemcpyDeviceToDevice, stream);
}

void topk_free(TopkWorkspace &ws)
{
    cudaFree(ws.keys);
    cudaFree(ws.cand_key);
    cudaFree(ws.cand_idx);
    cudaFree(ws.hist);
    cudaFree(ws.state);
    cudaFree(ws.block_counts);
    ws = TopkWorkspace();
}

}  // namespace dt
