// resolve_kernel.cu -- a9 / a2: the in-order containment resolve (Alg. 3 phase 3)
// and the phase-1 "is masked" filter on the GPU (R17, R18, R26).
//
//   kept(i) = score_i >= tau  and  no accepted box of the same strand contains (tpos_i, qpos_i),
// where "accepted" = boxes carried in from earlier windows + boxes kept at indices < i.
// Extensions never depend on the accepted set (R20), so only `kept` is recursive.  One warp walks
// the anchors 32 at a time ("serial over kept, parallel over covered"):
//   1. every lane tests its anchor against the ACTIVE accepted boxes (parallel over anchors);
//   2. the lowest still-undecided lane with score >= tau is kept; its box is broadcast and the
//      higher lanes test themselves against it; repeat (one round per kept anchor of the block).
// A box is active while it can still cover a future anchor: box.tend >= min tpos of all remaining
// anchors (an exact suffix minimum, so any anchor order is handled; for anchors sorted by target
// position the active list stays a handful of boxes).
#include "sfe_internal.cuh"

#define FULL 0xffffffffu

__global__ void block_min_kernel(const sfe_anchor *anchors, long long n, long long *blkmin)
{
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    long long v = (i < n) ? anchors[i].tpos : 0x7fffffffffffffffLL;
    for (int o = 16; o > 0; o >>= 1) { const long long y = __shfl_xor_sync(FULL, v, o); v = y < v ? y : v; }
    if ((threadIdx.x & 31) == 0 && i < n) blkmin[i >> 5] = v;
}

static __device__ __forceinline__ bool box_has(const sfe_box &b, long long t, long long q, int strand)
{
    return b.strand == strand && b.tstart <= t && t <= b.tend && b.qstart <= q && q <= b.qend;
}

// single warp
__global__ void resolve_kernel(const sfe_anchor *anchors, const sfe_result *results, long long n, int min_score,
                               sfe_box *accepted, long long accepted_cap, long long *n_accepted_io, uint8_t *keep,
                               sfe_stats *stats, long long *blkmin, sfe_box *act)
{
    const int lane = threadIdx.x & 31;
    const long long nblk = (n + 31) >> 5;
    // suffix minimum over block minima, in place (reverse order, 32 blocks per step)
    {
        long long carry = 0x7fffffffffffffffLL;
        for (long long hi = nblk; hi > 0; hi -= 32) {
            const long long b = hi - 1 - lane;
            long long v = (b >= 0) ? blkmin[b] : 0x7fffffffffffffffLL;
            for (int o = 1; o < 32; o <<= 1) { const long long y = __shfl_up_sync(FULL, v, o); if (lane >= o && y < v) v = y; }
            v = v < carry ? v : carry;
            if (b >= 0) blkmin[b] = v;
            carry = __shfl_sync(FULL, v, 31);
        }
    }
    long long nacc = *n_accepted_io;
    long long nact = 0;
    const bool commit = results != nullptr;
    // active list starts as every box carried in
    for (long long k = lane; k < nacc; k += 32) act[k] = accepted[k];
    nact = nacc;
    __syncwarp();
    long long c_kept = 0, c_cov = 0, c_below = 0;
    unsigned long long cells_tot = 0, cells_cov = 0;
    bool overflow = false;
    for (long long blk = 0; blk < nblk; blk++) {
        // retire boxes that end before every remaining anchor (stable in-place compaction)
        {
            const long long tmin = blkmin[blk];
            long long w = 0;
            for (long long base = 0; base < nact; base += 32) {
                const long long k = base + lane;
                sfe_box b; bool live = false;
                if (k < nact) { b = act[k]; live = b.tend >= tmin; }
                const unsigned m = __ballot_sync(FULL, live);
                if (live) act[w + __popc(m & ((1u << lane) - 1))] = b;
                w += __popc(m);
                __syncwarp();
            }
            nact = w;
        }
        const long long i = (blk << 5) + lane;
        const bool valid = i < n;
        long long tp = 0, qp = 0; int strand = 0, score = 0; unsigned long long cells = 0;
        sfe_box mine; mine.tstart = mine.tend = mine.qstart = mine.qend = 0; mine.strand = 0; mine.reserved = 0;
        if (valid) {
            tp = anchors[i].tpos; qp = anchors[i].qpos; strand = anchors[i].strand >= 0 ? 1 : -1;
            if (commit) {
                score = results[i].score; cells = results[i].cells;
                mine.tstart = results[i].tstart; mine.tend = results[i].tend;
                mine.qstart = results[i].qstart; mine.qend = results[i].qend; mine.strand = strand;
            }
        }
        bool cov = false;
        for (long long k = 0; k < nact; k++) { const sfe_box b = act[k]; cov = cov || box_has(b, tp, qp, strand); }
        cov = cov && valid;
        bool cand = valid && !cov && commit && score >= min_score;
        bool kept = false;
        unsigned mask = __ballot_sync(FULL, cand);
        while (mask) {
            const int leader = __ffs(mask) - 1;
            if (lane == leader) { kept = true; cand = false; }
            sfe_box lb;
            lb.tstart = __shfl_sync(FULL, mine.tstart, leader); lb.tend = __shfl_sync(FULL, mine.tend, leader);
            lb.qstart = __shfl_sync(FULL, mine.qstart, leader); lb.qend = __shfl_sync(FULL, mine.qend, leader);
            lb.strand = __shfl_sync(FULL, mine.strand, leader); lb.reserved = 0;
            if (valid && lane > leader && !cov && box_has(lb, tp, qp, strand)) { cov = true; cand = false; }
            if (lane == leader) {
                if (nacc < accepted_cap) { accepted[nacc] = lb; act[nact] = lb; }
            }
            if (nacc < accepted_cap) { nact++; } else overflow = true;
            nacc++;
            __syncwarp();
            mask = __ballot_sync(FULL, cand);
        }
        if (valid) {
            keep[i] = commit ? (cov ? 0 : (kept ? 1 : 2)) : (cov ? 0 : 1);
            c_kept += kept; c_cov += cov; c_below += (!cov && !kept);
            cells_tot += cells; if (cov) cells_cov += cells;
        }
    }
    for (int o = 16; o > 0; o >>= 1) {
        c_kept += __shfl_xor_sync(FULL, c_kept, o); c_cov += __shfl_xor_sync(FULL, c_cov, o);
        c_below += __shfl_xor_sync(FULL, c_below, o);
        cells_tot += __shfl_xor_sync(FULL, cells_tot, o); cells_cov += __shfl_xor_sync(FULL, cells_cov, o);
    }
    if (lane == 0) {
        if (commit) *n_accepted_io = overflow ? -nacc : nacc;   // negative: accepted_cap too small (needed -value)
        if (stats && commit) {
            stats->n_anchors += n; stats->n_kept += c_kept; stats->n_covered += c_cov; stats->n_below += c_below;
            stats->cells_total += cells_tot; stats->cells_covered += cells_cov;
        }
    }
}

int sfe_launch_resolve(const sfe_anchor *anchors, const sfe_result *results, long long n, int min_score, sfe_box *accepted,
                       long long accepted_cap, long long *n_accepted_io, uint8_t *keep, sfe_stats *stats, long long *blkmin,
                       sfe_box *act, cudaStream_t st)
{
    if (n <= 0) return SFE_OK;
    const int bs = 256;
    block_min_kernel<<<(unsigned)((n + bs - 1) / bs), bs, 0, st>>>(anchors, n, blkmin);
    resolve_kernel<<<1, 32, 0, st>>>(anchors, results, n, min_score, accepted, accepted_cap, n_accepted_io, keep, stats, blkmin, act);
    SFE_LAUNCH_CHECK();
}
