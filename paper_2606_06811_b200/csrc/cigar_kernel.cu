// cigar_kernel.cu -- a8, second part: join the two halves of every anchor and place the run-length
// CIGARs (R11, R12) at deterministic, anchor-ordered offsets of the caller's pool.
//
// The traceback walk itself happens inside ydrop_kernel (walk_traceback): the warp that computed a
// half walks its 4-bit pointers right away and stages the ops, in walk order (end cell -> origin),
// as a backward-linked list of segments in the ops arena.  What is left here is cheap and parallel:
//   join_kernel   one thread per anchor: score, box, cells, status, n_ops = n_ops(back) + n_ops(fwd);
//   scan_offsets  exclusive scan of n_ops in anchor order -> cigar_off;
//   emit_kernel   one warp per anchor copies the staged ops: the backward half's walk order (far end
//                 -> anchor) is already the output order, the forward half is reversed.
#include "sfe_internal.cuh"

__global__ void join_kernel(const sfe_anchor *anchors, const sfe_half *halves, long long n, const long long *sel,
                            long long n_sel, int want_cigar, sfe_result *results)
{
    const long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (x >= n_sel) return;
    const long long a = sel ? sel[x] : x;
    const sfe_half f = halves[2 * a], b = halves[2 * a + 1];
    const sfe_anchor an = anchors[a];
    sfe_result r;
    r.score_fwd = f.score; r.score_bwd = b.score; r.score = f.score + b.score;
    const uint32_t st = (f.status | b.status);
    r.tstart = an.tpos - b.end_j; r.tend = an.tpos + f.end_j;
    r.qstart = an.qpos - b.end_i; r.qend = an.qpos + f.end_i;
    r.cells = f.cells + b.cells;
    r.cigar_off = -1; r.n_ops = 0; r.n_ops_back = 0;
    if (want_cigar && !(st & (SFE_ST_PASS_OVERFLOW | SFE_ST_BAD_ANCHOR | SFE_ST_BAND_LIMIT | SFE_ST_SCORE_LIMIT | SFE_ST_INTERNAL))) {
        r.n_ops_back = b.n_ops; r.n_ops = b.n_ops + f.n_ops;
    }
    r.status = (st & 0xffu) | ((st & SFE_ST_PASS_OVERFLOW) ? SFE_ST_TB_OVERFLOW : 0u) |
               ((st & SFE_ST_OPS_OVERFLOW) ? SFE_ST_CIGAR_OVERFLOW : 0u);
    results[a] = r;
}

// exclusive scan of results[].n_ops into results[].cigar_off (single block, running carry).
// Anchors flagged SFE_ST_TB_OVERFLOW / SFE_ST_CIGAR_OVERFLOW keep cigar_off = -1 and contribute
// nothing in this pass; anchors that already have an offset (earlier pass) are skipped.
__global__ void scan_offsets_kernel(sfe_result *results, long long n, long long *pool_used, long long cap)
{
    __shared__ long long warp_sums[32];
    __shared__ long long carry;
    if (threadIdx.x == 0) carry = *pool_used;
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (long long base = 0; base < n; base += blockDim.x) {
        const long long i = base + threadIdx.x;
        long long v = 0;
        bool take = false;
        if (i < n) { take = results[i].n_ops > 0 && results[i].cigar_off < 0 && !(results[i].status & (SFE_ST_TB_OVERFLOW | SFE_ST_CIGAR_OVERFLOW)); v = take ? results[i].n_ops : 0; }
        long long incl = v;
        for (int o = 1; o < 32; o <<= 1) { const long long y = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += y; }
        if (lane == 31) warp_sums[wid] = incl;
        __syncthreads();
        if (wid == 0) {
            long long w = (lane < (blockDim.x >> 5)) ? warp_sums[lane] : 0, wi = w;
            for (int o = 1; o < 32; o <<= 1) { const long long y = __shfl_up_sync(0xffffffffu, wi, o); if (lane >= o) wi += y; }
            warp_sums[lane] = wi - w;
        }
        __syncthreads();
        const long long off = carry + warp_sums[wid] + incl - v;
        if (take) {
            if (off + v <= cap) results[i].cigar_off = off;
            else results[i].status |= SFE_ST_CIGAR_OVERFLOW;
        }
        __syncthreads();
        if (threadIdx.x == blockDim.x - 1) carry = off + v;
        __syncthreads();
    }
    if (threadIdx.x == 0) *pool_used = carry;
}

// Copy one half's staged ops.  The segments form a backward-linked list; the last one holds the walk
// indices [n - count, n).  dir = +1: walk index x goes to dst[x]; dir = -1: to dst[n - 1 - x].
static __device__ void copy_half_ops(const sfe_half &h, const uint32_t *stage, uint32_t *dst, int dir, int lane)
{
    int hi = h.n_ops;
    uint32_t seg = h.ops_seg;
    while (seg != SFE_NO_SEG && hi > 0) {
        const uint32_t prev = stage[seg];
        const int cnt = (int)stage[seg + 1];
        const int lo = hi - cnt;
        for (int x = lane; x < cnt; x += 32) {
            const int w = lo + x;
            dst[dir > 0 ? w : h.n_ops - 1 - w] = stage[seg + 2 + x];
        }
        hi = lo; seg = prev;
    }
}

__global__ void emit_kernel(const sfe_half *halves, long long n, const long long *sel, long long n_sel,
                            const uint32_t *stage, const sfe_result *results, uint32_t *cigar_pool)
{
    const long long x = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (x >= n_sel) return;
    const long long a = sel ? sel[x] : x;
    const sfe_result r = results[a];
    if (r.n_ops <= 0 || r.cigar_off < 0 || (r.status & (SFE_ST_CIGAR_OVERFLOW | SFE_ST_TB_OVERFLOW))) return;
    uint32_t *dst = cigar_pool + r.cigar_off;
    copy_half_ops(halves[2 * a + 1], stage, dst, +1, lane);
    copy_half_ops(halves[2 * a], stage, dst + r.n_ops_back, -1, lane);
}

int sfe_launch_join(const sfe_anchor *anchors, const sfe_half *halves, long long n, const long long *sel, long long n_sel,
                    int want_cigar, sfe_result *results, cudaStream_t st)
{
    if (n_sel <= 0) return SFE_OK;
    const int bs = 128;
    SFE_KL join_kernel<<<(unsigned)((n_sel + bs - 1) / bs), bs, 0, st>>>(anchors, halves, n, sel, n_sel, want_cigar, results);
    SFE_LAUNCH_CHECK();
}

int sfe_launch_scan_emit(const sfe_half *halves, long long n, const long long *sel, long long n_sel, const uint32_t *stage,
                         sfe_result *results, uint32_t *cigar_pool, long long cap, long long *pool_used, cudaStream_t st)
{
    if (n <= 0) return SFE_OK;
    SFE_KL scan_offsets_kernel<<<1, 1024, 0, st>>>(results, n, pool_used, cap);
    if (n_sel > 0) {
        const int bs = 256;                                   // 8 anchors per block, one warp each
        SFE_KL emit_kernel<<<(unsigned)((n_sel * 32 + bs - 1) / bs), bs, 0, st>>>(halves, n, sel, n_sel, stage, results, cigar_pool);
    }
    SFE_LAUNCH_CHECK();
}
