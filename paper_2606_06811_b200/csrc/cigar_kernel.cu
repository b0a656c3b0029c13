// cigar_kernel.cu -- a8: join the two halves of every anchor and emit run-length CIGARs by walking
// the 4-bit traceback pointers that ydrop_kernel spilled to the HBM arena (R11, R12).
//
// Pass 1 (join_count): one thread per anchor joins the halves into sfe_result (score, box, cells,
// status) and, if a CIGAR is wanted, walks both halves once to count their runs.
// An exclusive scan over n_ops gives deterministic pool offsets in anchor order.
// Pass 2 (emit): the same walk again, writing ops.  The backward half's walk order (far end ->
// anchor) is already the output order; the forward half is written from the end of its slot.
#include "sfe_internal.cuh"

#define ST_PASS_OVERFLOW 0x100u

struct TbCursor {          // random access to a half's records, cheap for monotonically decreasing indices
    const uint32_t *pool; const int32_t *chunk_prev;
    int chunk, ord;        // current chunk id and its ordinal in the half's list
    int last_chunk, last_ord;
    __device__ __forceinline__ const uint32_t *rec(int ridx)
    {
        const int o = ridx / SFE_CHUNK_RECS;
        if (o > ord) { chunk = last_chunk; ord = last_ord; }   // rare: header / record straddle a chunk edge
        while (ord > o) { chunk = chunk_prev[chunk]; ord--; }
        return pool + ((size_t)chunk * SFE_CHUNK_RECS + (ridx - o * SFE_CHUNK_RECS)) * 32;
    }
};

// Walk one half from its end cell to the origin.  EMIT == false: returns the number of runs.
// EMIT == true: writes runs; step = +1 writes dst[0], dst[1], ... in walk order, step = -1 writes
// dst[0], dst[-1], ...
template <bool EMIT>
static __device__ int walk_half(const sfe_half &h, const uint32_t *pool, const int32_t *chunk_prev, uint32_t *dst, int step)
{
    if (h.end_i == 0 && h.end_j == 0) return 0;
    TbCursor cur; cur.pool = pool; cur.chunk_prev = chunk_prev; cur.chunk = h.last_chunk;
    cur.ord = (h.n_rec - 1) / SFE_CHUNK_RECS;
    cur.last_chunk = cur.chunk; cur.last_ord = cur.ord;
    // locate the header of the strip holding the end row
    int strip = h.n_strips - 1, hdr = h.last_hdr;
    int i = h.end_i, j = h.end_j;
    const uint32_t *hr = cur.rec(hdr);
    while (strip > (i >> 5)) { hdr = (int)hr[1]; strip--; hr = cur.rec(hdr); }
    int cs = (int)hr[0], prev_hdr = (int)hr[1];
    int state = 0, cur_op = -1, run = 0, nruns = 0;
    while (!(i == 0 && j == 0 && state == 0)) {
        if ((i >> 5) < strip) {                     // crossed into the strip above
            hdr = prev_hdr; strip--;
            hr = cur.rec(hdr); cs = (int)hr[0]; prev_hdr = (int)hr[1];
        }
        const int lane = i & 31;
        const int t = j - cs + lane;
        const uint32_t w = cur.rec(hdr + 1 + (t >> 3))[lane];
        const uint32_t nib = (w >> ((7 - (t & 7)) * 4)) & 15u;   // bit3 !M, bit2 !E, bit1 E ext, bit0 F ext
        int op = -1;
        if (state == 0) {
            if (!(nib & 8u)) { op = SFE_OP_M; i--; j--; }
            else state = (nib & 4u) ? 2 : 1;
        } else if (state == 1) {
            op = SFE_OP_I; i--; if (!(nib & 2u)) state = 0;
        } else {
            op = SFE_OP_D; j--; if (!(nib & 1u)) state = 0;
        }
        if (op >= 0) {
            if (op == cur_op) run++;
            else {
                if (cur_op >= 0) { if (EMIT) { *dst = ((uint32_t)run << 4) | (uint32_t)cur_op; dst += step; } nruns++; }
                cur_op = op; run = 1;
            }
        }
    }
    if (cur_op >= 0) { if (EMIT) { *dst = ((uint32_t)run << 4) | (uint32_t)cur_op; } nruns++; }
    return nruns;
}

__global__ void join_count_kernel(const sfe_anchor *anchors, const sfe_half *halves, long long n, const long long *sel,
                                  long long n_sel, const uint32_t *pool, const int32_t *chunk_prev, int want_cigar,
                                  sfe_result *results, int32_t *nops_fwd)
{
    const long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (x >= n_sel) return;
    const long long a = sel ? sel[x] : x;
    const sfe_half f = halves[2 * a], b = halves[2 * a + 1];
    const sfe_anchor an = anchors[a];
    sfe_result r;
    r.score_fwd = f.score; r.score_bwd = b.score; r.score = f.score + b.score;
    uint32_t st = (f.status | b.status);
    r.tstart = an.tpos - b.end_j; r.tend = an.tpos + f.end_j;
    r.qstart = an.qpos - b.end_i; r.qend = an.qpos + f.end_i;
    r.cells = f.cells + b.cells;
    r.cigar_off = -1; r.n_ops = 0; r.n_ops_back = 0;
    int nf = 0;
    if (want_cigar && !(st & (ST_PASS_OVERFLOW | SFE_ST_BAD_ANCHOR | SFE_ST_BAND_LIMIT))) {
        const int nb = walk_half<false>(b, pool, chunk_prev, nullptr, 0);
        nf = walk_half<false>(f, pool, chunk_prev, nullptr, 0);
        r.n_ops_back = nb; r.n_ops = nb + nf;
    }
    r.status = (st & 0xffu) | ((st & ST_PASS_OVERFLOW) ? SFE_ST_TB_OVERFLOW : 0u);
    results[a] = r;
    if (nops_fwd) nops_fwd[a] = nf;
}

// exclusive scan of results[].n_ops into results[].cigar_off (single block, running carry).
// Anchors flagged SFE_ST_TB_OVERFLOW keep cigar_off = -1 and contribute nothing in this pass.
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

__global__ void emit_kernel(const sfe_half *halves, long long n, const long long *sel, long long n_sel, const uint32_t *pool,
                            const int32_t *chunk_prev, const sfe_result *results, uint32_t *cigar_pool)
{
    const long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (x >= n_sel) return;
    const long long a = sel ? sel[x] : x;
    const sfe_result r = results[a];
    if (r.n_ops <= 0 || r.cigar_off < 0 || (r.status & (SFE_ST_CIGAR_OVERFLOW | SFE_ST_TB_OVERFLOW))) return;
    uint32_t *dst = cigar_pool + r.cigar_off;
    walk_half<true>(halves[2 * a + 1], pool, chunk_prev, dst, +1);
    walk_half<true>(halves[2 * a], pool, chunk_prev, dst + r.n_ops - 1, -1);
}

int sfe_launch_join(const sfe_anchor *anchors, const sfe_half *halves, long long n, const long long *sel, long long n_sel,
                    const uint32_t *pool, const int32_t *chunk_prev, int want_cigar, sfe_result *results, cudaStream_t st)
{
    if (n_sel <= 0) return SFE_OK;
    const int bs = 128;
    join_count_kernel<<<(unsigned)((n_sel + bs - 1) / bs), bs, 0, st>>>(anchors, halves, n, sel, n_sel, pool, chunk_prev,
                                                                     want_cigar, results, nullptr);
    SFE_LAUNCH_CHECK();
}

int sfe_launch_scan_emit(const sfe_half *halves, long long n, const long long *sel, long long n_sel, const uint32_t *pool,
                         const int32_t *chunk_prev, sfe_result *results, uint32_t *cigar_pool, long long cap,
                         long long *pool_used, cudaStream_t st)
{
    if (n <= 0) return SFE_OK;
    scan_offsets_kernel<<<1, 1024, 0, st>>>(results, n, pool_used, cap);
    if (n_sel > 0) {
        const int bs = 128;
        emit_kernel<<<(unsigned)((n_sel + bs - 1) / bs), bs, 0, st>>>(halves, n, sel, n_sel, pool, chunk_prev, results, cigar_pool);
    }
    SFE_LAUNCH_CHECK();
}
