// queue_kernels.cu -- a3: length-binned ticket order for the persistent work queue, the free-chunk ring of the
// traceback arena and the overflow re-run selection.
#include "sfe_internal.cuh"


// ---- a3: bins -----------------------------------------------------------------------------------
// Length proxy of a half = min(rows available, columns available) to the pair's limit
// (the true length is unknown a priori).  Bin = floor(log2(proxy + 1)); tickets are
// issued longest bin first so that the heavy tail starts early ("presorting ... by
// length and deploying persistent thread queues").
static __device__ __forceinline__ int half_bin(const sfe_anchor &an, const sfe_pair *pairs, int n_pairs, long long q_len, int dir)
{
    if (an.pair < 0 || an.pair >= n_pairs) return 0;
    const sfe_pair pr = pairs[an.pair];
    long long qb = pr.q_begin, qe = pr.q_end;
    if (an.strand < 0) { qb = q_len - pr.q_end; qe = q_len - pr.q_begin; }
    long long n = dir == 0 ? qe - an.qpos : an.qpos - qb;
    long long m = dir == 0 ? pr.t_end - an.tpos : an.tpos - pr.t_begin;
    long long v = n < m ? n : m;
    if (v < 0) v = 0;
    if (v > 0x3fffffff) v = 0x3fffffff;
    return 31 - __clz((int)v + 1);                   // 0..30
}

// prio (may be NULL): one byte per anchor.  0 = bin by the proxy.  p > 0 = bin 31 + p, i.e. before every proxy-binned
// ticket and ordered among themselves by p: sfe_speculate passes 1 for predicted leaders with followers ("long-likely";
// in a genome-scale pair the distance to the pair's end says nothing: every anchor is far from it) and
// 1 + floor(log2(span)) for the kept anchors' traceback batch, whose extensions are already known.
__global__ void bin_count_kernel(const sfe_anchor *anchors, long long n_anchors, const sfe_pair *pairs, int n_pairs,
                                 long long q_len, const uint8_t *prio, unsigned int *hist)
{
    const long long h = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (h >= 2 * n_anchors) return;
    const int pb = prio ? prio[h >> 1] : 0;
    atomicAdd(&hist[pb ? min(63, 31 + pb) : half_bin(anchors[h >> 1], pairs, n_pairs, q_len, (int)(h & 1))], 1u);
}

// hist[0..63] -> hist[64..127] = start offset of each bin in descending-bin order
__global__ void bin_offsets_kernel(unsigned int *hist)
{
    if (threadIdx.x == 0) {
        unsigned int off = 0;
        for (int b = 63; b >= 0; b--) { hist[64 + b] = off; off += hist[b]; }
    }
}

__global__ void bin_scatter_kernel(const sfe_anchor *anchors, long long n_anchors, const sfe_pair *pairs, int n_pairs,
                                   long long q_len, const uint8_t *prio, unsigned int *hist, int32_t *tickets)
{
    const long long h = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (h >= 2 * n_anchors) return;
    const int pb = prio ? prio[h >> 1] : 0;
    const int b = pb ? min(63, 31 + pb) : half_bin(anchors[h >> 1], pairs, n_pairs, q_len, (int)(h & 1));
    tickets[atomicAdd(&hist[64 + b], 1u)] = (int32_t)h;
}

// How many of the longest-first tickets go to the cooperative row kernel (ydrop_row_kernel.cu): the priority bins
// (32..63: long-likely leaders / known long extensions) if there are any, up to cap_prio; else whole proxy bins from the top
// while they hold at most cap_plain tickets and promise at least 2^min_bin rows.  One CTA works on one such half.
__global__ void row_split_kernel(const unsigned int *hist, unsigned long long *counters, unsigned int cap_prio, unsigned int cap_plain,
                                 int min_bin)
{
    if (threadIdx.x != 0) return;
    unsigned int n = 0;
    for (int b = 63; b >= 32; b--) n += hist[b];
    if (n > 0) { counters[CNT_ROW_N] = n < cap_prio ? n : cap_prio; return; }
    for (int b = 31; b >= min_bin; b--) {
        if (n + hist[b] > cap_plain) break;
        n += hist[b];
    }
    counters[CNT_ROW_N] = n;
}

__global__ void iota_tickets_kernel(int32_t *tickets, long long n)
{
    const long long h = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (h < n) tickets[h] = (int32_t)h;
}

int sfe_launch_tickets(const sfe_anchor *anchors, long long n_anchors, const sfe_pair *pairs, int n_pairs, long long q_len,
                       bool binned, const uint8_t *prio, unsigned int *hist, int32_t *tickets, unsigned long long *counters,
                       long long cap_prio, long long cap_plain, cudaStream_t st)
{
    const long long n = 2 * n_anchors;
    if (n <= 0) return SFE_OK;
    const int bs = 256;
    const unsigned nb = (unsigned)((n + bs - 1) / bs);
    if (!binned) SFE_KL iota_tickets_kernel<<<nb, bs, 0, st>>>(tickets, n);
    else {
        if (cudaMemsetAsync(hist, 0, 128 * sizeof(unsigned int), st) != cudaSuccess) return SFE_ECUDA;
        SFE_KL bin_count_kernel<<<nb, bs, 0, st>>>(anchors, n_anchors, pairs, n_pairs, q_len, prio, hist);
        SFE_KL bin_offsets_kernel<<<1, 32, 0, st>>>(hist);
        SFE_KL bin_scatter_kernel<<<nb, bs, 0, st>>>(anchors, n_anchors, pairs, n_pairs, q_len, prio, hist, tickets);
        if (cap_prio > 0 || cap_plain > 0) SFE_KL row_split_kernel<<<1, 32, 0, st>>>(hist, counters, (unsigned int)cap_prio, (unsigned int)cap_plain, 12);
    }
    SFE_LAUNCH_CHECK();
}

// ---- free-chunk ring of the traceback arena (sfe_internal.cuh: SfeFreeRing) ------------------------
__global__ void ring_init_kernel(int32_t *ring, SfeFreeRing *st, int n_chunks)
{
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i < n_chunks) ring[i] = (int32_t)i;
    if (i == 0) { st->head = 0ULL; st->tail = (unsigned long long)n_chunks; st->avail = n_chunks; }
}

int sfe_launch_ring_init(int32_t *ring, SfeFreeRing *st, int n_chunks, cudaStream_t stream)
{
    const int bs = 256;
    SFE_KL ring_init_kernel<<<(unsigned)((n_chunks + bs - 1) / bs), bs, 0, stream>>>(ring, st, n_chunks);
    SFE_LAUNCH_CHECK();
}

// ---- overflow re-run selection --------------------------------------------------------------------
// Anchors with a half whose traceback did not fit in this pass: append to sel[], and make tickets.
// A half that overflowed went on score-only to its end, so the chunks it needs are known exactly:
// one record per strip header and per 16 steps.  Halves that need more than the whole arena are
// not selected (their anchor keeps SFE_ST_TB_OVERFLOW); the largest need goes to counters[CNT_MAXNEED].
static __device__ __forceinline__ long long half_need_chunks(const sfe_half &h)
{
    const long long recs = (long long)h.n_strips + (long long)h.steps / 16 + 2;
    return (recs + SFE_CHUNK_RECS - 1) / SFE_CHUNK_RECS;
}

__global__ void select_overflow_kernel(const sfe_half *halves, long long n_anchors, long long *sel, int32_t *tickets,
                                       unsigned long long *counters, int n_chunks)
{
    const long long a = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (a >= n_anchors) return;
    if ((halves[2 * a].status | halves[2 * a + 1].status) & SFE_ST_PASS_OVERFLOW) {
        const long long n0 = half_need_chunks(halves[2 * a]), n1 = half_need_chunks(halves[2 * a + 1]);
        const long long need = n0 > n1 ? n0 : n1;
        if (need > n_chunks) return;
        atomicMax(&counters[CNT_MAXNEED], (unsigned long long)need);
        const unsigned long long k = atomicAdd(&counters[CNT_RERUN], 1ULL);
        sel[k] = a; tickets[2 * k] = (int32_t)(2 * a); tickets[2 * k + 1] = (int32_t)(2 * a + 1);
    }
}

int sfe_launch_select_overflow(const sfe_half *halves, long long n_anchors, long long *sel, int32_t *tickets,
                               unsigned long long *counters, int n_chunks, cudaStream_t st)
{
    const int bs = 256;
    SFE_KL select_overflow_kernel<<<(unsigned)((n_anchors + bs - 1) / bs), bs, 0, st>>>(halves, n_anchors, sel, tickets, counters, n_chunks);
    SFE_LAUNCH_CHECK();
}
