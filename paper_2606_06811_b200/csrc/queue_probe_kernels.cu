// queue_probe_kernels.cu -- a3: length-binned ticket order for the persistent work queue, the
// overflow re-run selection, and the integer-issue microbenchmark used for the roofline (8(d)).
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

__global__ void bin_count_kernel(const sfe_anchor *anchors, long long n_anchors, const sfe_pair *pairs, int n_pairs,
                                 long long q_len, unsigned int *hist)
{
    const long long h = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (h >= 2 * n_anchors) return;
    atomicAdd(&hist[half_bin(anchors[h >> 1], pairs, n_pairs, q_len, (int)(h & 1))], 1u);
}

// hist[0..31] -> hist[32..63] = start offset of each bin in descending-bin order
__global__ void bin_offsets_kernel(unsigned int *hist)
{
    if (threadIdx.x == 0) {
        unsigned int off = 0;
        for (int b = 31; b >= 0; b--) { hist[32 + b] = off; off += hist[b]; }
    }
}

__global__ void bin_scatter_kernel(const sfe_anchor *anchors, long long n_anchors, const sfe_pair *pairs, int n_pairs,
                                   long long q_len, unsigned int *hist, int32_t *tickets)
{
    const long long h = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (h >= 2 * n_anchors) return;
    const int b = half_bin(anchors[h >> 1], pairs, n_pairs, q_len, (int)(h & 1));
    tickets[atomicAdd(&hist[32 + b], 1u)] = (int32_t)h;
}

__global__ void iota_tickets_kernel(int32_t *tickets, long long n)
{
    const long long h = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (h < n) tickets[h] = (int32_t)h;
}

int sfe_launch_tickets(const sfe_anchor *anchors, long long n_anchors, const sfe_pair *pairs, int n_pairs, long long q_len,
                       bool binned, unsigned int *hist, int32_t *tickets, cudaStream_t st)
{
    const long long n = 2 * n_anchors;
    if (n <= 0) return SFE_OK;
    const int bs = 256;
    const unsigned nb = (unsigned)((n + bs - 1) / bs);
    if (!binned) iota_tickets_kernel<<<nb, bs, 0, st>>>(tickets, n);
    else {
        if (cudaMemsetAsync(hist, 0, 64 * sizeof(unsigned int), st) != cudaSuccess) return SFE_ECUDA;
        bin_count_kernel<<<nb, bs, 0, st>>>(anchors, n_anchors, pairs, n_pairs, q_len, hist);
        bin_offsets_kernel<<<1, 32, 0, st>>>(hist);
        bin_scatter_kernel<<<nb, bs, 0, st>>>(anchors, n_anchors, pairs, n_pairs, q_len, hist, tickets);
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
    ring_init_kernel<<<(unsigned)((n_chunks + bs - 1) / bs), bs, 0, stream>>>(ring, st, n_chunks);
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
    select_overflow_kernel<<<(unsigned)((n_anchors + bs - 1) / bs), bs, 0, st>>>(halves, n_anchors, sel, tickets, counters, n_chunks);
    SFE_LAUNCH_CHECK();
}

// ---- integer-issue microbenchmark ---------------------------------------------------------------------
// Register-only loops of independent chains, one kernel per opcode mix, at full occupancy.  Each
// iteration issues OPS instructions per thread (checked against cuobjdump: DESIGN.md "Roofline").
#define PROBE_CHAINS 8
template <int MIX>
__global__ void __launch_bounds__(256) probe_kernel(int iters, int seed, int *sink)
{
    int a[PROBE_CHAINS], b[PROBE_CHAINS];
#pragma unroll
    for (int c = 0; c < PROBE_CHAINS; c++) { a[c] = seed + threadIdx.x * (c + 1); b[c] = seed ^ (c * 77 + blockIdx.x); }
    const int k1 = seed | 1, k2 = seed + 3;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int c = 0; c < PROBE_CHAINS; c++) {
            if (MIX == 1) {            // ALU pipe only: SHF + LOP3 (an add.s32 would become IMAD.IADD on the FMA pipe)
                asm volatile("shf.l.wrap.b32 %0, %0, %1, 3;" : "+r"(a[c]) : "r"(b[c]));
                asm volatile("xor.b32 %0, %0, %1;" : "+r"(b[c]) : "r"(a[c]));
            } else if (MIX == 2) {     // DPX: VIADDMNMX + VIMNMX3
                a[c] = __viaddmax_s32(a[c], k1, b[c]);
                b[c] = __vimax3_s32(b[c], a[c], k2);
            } else if (MIX == 3) {     // FMA pipe: IMAD
                asm volatile("mad.lo.s32 %0, %0, %1, %2;" : "+r"(a[c]) : "r"(k1), "r"(b[c]));
                asm volatile("mad.lo.s32 %0, %0, %1, %2;" : "+r"(b[c]) : "r"(k2), "r"(a[c]));
            } else {                   // mixed: one ALU/DPX op + one IMAD (both pipes busy)
                a[c] = __viaddmax_s32(a[c], k1, b[c]);
                asm volatile("mad.lo.s32 %0, %0, %1, %2;" : "+r"(b[c]) : "r"(k2), "r"(a[c]));
            }
        }
    }
    int r = 0;
#pragma unroll
    for (int c = 0; c < PROBE_CHAINS; c++) r ^= a[c] ^ b[c];
    if (r == 0x7fffabcd) *sink = r;
}

int sfe_launch_probe(int mix, int iters, int blocks, int *sink, cudaStream_t st)
{
    switch (mix) {
    case 1: probe_kernel<1><<<blocks, 256, 0, st>>>(iters, 12345, sink); break;
    case 2: probe_kernel<2><<<blocks, 256, 0, st>>>(iters, 12345, sink); break;
    case 3: probe_kernel<3><<<blocks, 256, 0, st>>>(iters, 12345, sink); break;
    default: probe_kernel<0><<<blocks, 256, 0, st>>>(iters, 12345, sink); break;
    }
    SFE_LAUNCH_CHECK();
}
