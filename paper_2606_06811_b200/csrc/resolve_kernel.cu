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
#define RES_ACT_S 64                  // active boxes mirrored in shared memory by resolve_kernel

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

// Decide one block of 32 anchors in anchor order (whole warp).  live = valid and not covered by an older box;
// cand = live and score >= tau.  kept(l) = cand(l) and no kept lower lane's box contains l's point.
// Only a candidate whose box reaches the smallest tpos among the later live lanes can cover anybody in the
// block ("reaching").  The reaching candidates are visited in lane order: one that is already covered is not
// kept and covers nobody; otherwise it is kept and every later live lane tests itself against its box in
// parallel.  Rounds <= kept reaching candidates (none for disjoint boxes such as C4's); the non-reaching
// candidates are kept iff nothing covered them.  Returns the kept mask; cov is updated for every live lane
// (candidate or below tau: R17 is tested before R16).
static __device__ unsigned decide_block(bool valid, bool live, bool cand, bool &cov, const sfe_box &mine, long long tp, long long qp, int strand,
                                        int lane)
{
    __shared__ sfe_box sb[32];
    __syncwarp();
    sb[lane] = mine;
    __syncwarp();                                                 // the boxes are read by other lanes below
    // `after` = a lower bound of the tpos of every later live lane.  Sorted block (the normal case): the next lane's tpos;
    // otherwise the exact suffix minimum over live lanes.  (A smaller bound only adds rounds, never changes a decision.)
    const long long tpv = valid ? tp : 0x7fffffffffffffffLL;      // (covered lanes count too: still a lower bound)
    long long after = __shfl_down_sync(FULL, tpv, 1);
    if (lane == 31) after = 0x7fffffffffffffffLL;
    if (!__all_sync(FULL, after >= tpv)) {                        // not sorted: the block's anchors are not in position order
        long long suf = live ? tp : 0x7fffffffffffffffLL;         // inclusive suffix minimum of tpos over live lanes
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const long long y = __shfl_down_sync(FULL, suf, o); if (lane + o < 32 && y < suf) suf = y; }
        after = __shfl_down_sync(FULL, suf, 1);
        if (lane == 31) after = 0x7fffffffffffffffLL;
    }
    const unsigned reach = __ballot_sync(FULL, cand && mine.tend >= after);
    unsigned covm = 0;
    for (unsigned m = reach; m; m &= m - 1) {
        const int l = __ffs(m) - 1;
        if ((covm >> l) & 1u) continue;
        const sfe_box b = sb[l];
        covm |= __ballot_sync(FULL, live && lane > l && box_has(b, tp, qp, strand));
    }
    if ((covm >> lane) & 1u) cov = true;
    return __ballot_sync(FULL, cand && !((covm >> lane) & 1u));
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
    // The warp is latency-bound, so: the next block's anchors / results are loaded one iteration ahead, the first
    // RES_ACT_S active boxes are mirrored in shared memory (retire pass and cover scan read the mirror).
    __shared__ sfe_box act_s[RES_ACT_S];
    for (long long k = lane; k < nacc; k += 32) { const sfe_box b = accepted[k]; act[k] = b; if (k < RES_ACT_S) act_s[k] = b; }
    nact = nacc;
    __syncwarp();
    long long c_kept = 0, c_cov = 0, c_below = 0;
    unsigned long long cells_tot = 0, cells_cov = 0;
    bool overflow = false;
    struct Item { long long tp, qp, tmin; int strand, score; unsigned long long cells; sfe_box box; bool valid; };
    auto load_item = [&](long long blk) {
        Item it;
        const long long i = (blk << 5) + lane;
        it.valid = i < n; it.tp = 0; it.qp = 0; it.strand = 0; it.score = 0; it.cells = 0;
        it.box.tstart = it.box.tend = it.box.qstart = it.box.qend = 0; it.box.strand = 0; it.box.reserved = 0;
        it.tmin = blkmin[blk];
        if (it.valid) {
            const sfe_anchor an = anchors[i];
            it.tp = an.tpos; it.qp = an.qpos; it.strand = an.strand >= 0 ? 1 : -1;
            if (commit) {
                const sfe_result r = results[i];
                it.score = r.score; it.cells = r.cells;
                it.box.tstart = r.tstart; it.box.tend = r.tend; it.box.qstart = r.qstart; it.box.qend = r.qend; it.box.strand = it.strand;
            }
        }
        return it;
    };
    Item nxt = load_item(0);
    for (long long blk = 0; blk < nblk; blk++) {
        const Item cur = nxt;
        if (blk + 1 < nblk) nxt = load_item(blk + 1);
        if (nact > 0) {                                   // retire boxes that end before every remaining anchor (stable compaction)
            long long w = 0;
            const bool from_s = nact <= RES_ACT_S;
            for (long long base = 0; base < nact; base += 32) {
                const long long k = base + lane;
                sfe_box b; bool live = false;
                if (k < nact) { b = from_s ? act_s[k] : act[k]; live = b.tend >= cur.tmin; }
                const unsigned m = __ballot_sync(FULL, live);
                __syncwarp();
                if (live) { const long long d = w + __popc(m & ((1u << lane) - 1)); act[d] = b; if (d < RES_ACT_S) act_s[d] = b; }
                w += __popc(m);
                __syncwarp();
            }
            nact = w;
        }
        const long long i = (blk << 5) + lane;
        const bool valid = cur.valid;
        const long long tp = cur.tp, qp = cur.qp; const int strand = cur.strand, score = cur.score;
        const unsigned long long cells = cur.cells;
        const sfe_box mine = cur.box;
        bool cov = false;
        const long long ns = nact < RES_ACT_S ? nact : RES_ACT_S;
        for (long long k = 0; k < ns; k++) { const sfe_box b = act_s[k]; cov = cov || box_has(b, tp, qp, strand); }
        for (long long k = ns; k < nact; k++) { const sfe_box b = act[k]; cov = cov || box_has(b, tp, qp, strand); }
        cov = cov && valid;
        const bool live = valid && !cov, cand = live && commit && score >= min_score;
        const unsigned kmask = decide_block(valid, live, cand, cov, mine, tp, qp, strand, lane);
        const bool kept = (kmask >> lane) & 1u;
        if (kept) {                                               // append the kept boxes in lane order
            const long long r = __popc(kmask & ((1u << lane) - 1));
            if (nacc + r < accepted_cap) { accepted[nacc + r] = mine; act[nact + r] = mine; if (nact + r < RES_ACT_S) act_s[nact + r] = mine; }
        }
        {
            const long long nk = __popc(kmask);
            const long long fit = nacc + nk <= accepted_cap ? nk : (accepted_cap > nacc ? accepted_cap - nacc : 0);
            if (fit < nk) overflow = true;
            nact += fit; nacc += nk;
        }
        __syncwarp();
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
            stats->n_extended += n; stats->n_windows += 1;
        }
    }
}

int sfe_launch_resolve(const sfe_anchor *anchors, const sfe_result *results, long long n, int min_score, sfe_box *accepted,
                       long long accepted_cap, long long *n_accepted_io, uint8_t *keep, sfe_stats *stats, long long *blkmin,
                       sfe_box *act, cudaStream_t st)
{
    if (n <= 0) return SFE_OK;
    const int bs = 256;
    SFE_KL block_min_kernel<<<(unsigned)((n + bs - 1) / bs), bs, 0, st>>>(anchors, n, blkmin);
    SFE_KL resolve_kernel<<<1, 32, 0, st>>>(anchors, results, n, min_score, accepted, accepted_cap, n_accepted_io, keep, stats, blkmin, act);
    SFE_LAUNCH_CHECK();
}

// =====================================================================================================
// Algorithm 3 as a device-side loop: sfe_speculate's three phases per window.
//   spec_scan    phase 1: from the cursor, test anchors against the ACTIVE accepted boxes;
//                covered anchors are final (the accepted set only grows): keep = 0, result = "skipped";
//                the first K uncovered anchors become the window (their indices and a compact copy).
//   (phase 2 = sfe_ydrop_batch on the compact window)
//   spec_commit  phase 3: in window order, the resolve rule against the boxes kept
//                earlier IN THIS WINDOW (older boxes were already tested by the scan); results and keep
//                flags are scattered back to anchor order; kept boxes join `accepted` and the active list.
// The active list persists across windows in device memory; a box leaves it when its tend is below the
// suffix minimum of tpos over all anchors not yet scanned (exact for any anchor order).
// =====================================================================================================
struct SpecState { long long cursor, win_n, nact, nacc, overflow; };

__global__ void suffix_min_kernel(long long *blkmin, long long nblk)
{
    const int lane = threadIdx.x & 31;
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

__global__ void spec_init_kernel(SpecState *st, const sfe_box *accepted, const long long *n_accepted, sfe_box *act)
{
    const int lane = threadIdx.x & 31;
    const long long nacc = *n_accepted;
    for (long long k = lane; k < nacc; k += 32) act[k] = accepted[k];
    if (lane == 0) { st->cursor = 0; st->win_n = 0; st->nact = nacc; st->nacc = nacc; st->overflow = 0; }
}

// stable in-place compaction of the live boxes (tend >= tmin); returns the new count (whole warp)
static __device__ long long retire_boxes(sfe_box *act, long long nact, long long tmin, int lane)
{
    long long w = 0;
    for (long long base = 0; base < nact; base += 32) {
        const long long k = base + lane;
        sfe_box b; bool live = false;
        if (k < nact) { b = act[k]; live = b.tend >= tmin; }
        const unsigned m = __ballot_sync(FULL, live);
        __syncwarp();
        if (live) act[w + __popc(m & ((1u << lane) - 1))] = b;
        w += __popc(m);
        __syncwarp();
    }
    return w;
}

// single warp
__global__ void spec_scan_kernel(SpecState *st, const sfe_anchor *anchors, long long n, const long long *blkmin, long long K,
                                 sfe_box *act, long long *win_idx, sfe_anchor *win_anchors, uint8_t *keep,
                                 sfe_result *results, sfe_stats *stats)
{
    const int lane = threadIdx.x & 31;
    long long j = st->cursor, nact = st->nact, wn = 0, c_cov = 0;
    while (j < n && wn < K) {
        const long long blk = j >> 5;
        nact = retire_boxes(act, nact, blkmin[blk], lane);
        const long long i = (blk << 5) + lane;
        const bool valid = i >= j && i < n;
        long long tp = 0, qp = 0; int strand = 0;
        sfe_anchor an;
        if (valid) { an = anchors[i]; tp = an.tpos; qp = an.qpos; strand = an.strand >= 0 ? 1 : -1; }
        bool cov = false;
        for (long long k = 0; k < nact; k++) { const sfe_box b = act[k]; cov = cov || box_has(b, tp, qp, strand); }
        cov = cov && valid;
        const unsigned um = __ballot_sync(FULL, valid && !cov);
        const int rank = __popc(um & ((1u << lane) - 1));
        // take uncovered anchors in order until the window is full; the cursor stops after the last one taken
        const long long room = K - wn;
        const int n_unc = __popc(um);
        long long next_j = ((blk + 1) << 5) < n ? ((blk + 1) << 5) : n;
        if (n_unc > room) {
            // the (room+1)-th uncovered lane and everything after it stay for the next window
            unsigned m = um; int stop_lane = 0;
            for (long long r = 0; r <= room; r++) { stop_lane = __ffs(m) - 1; m &= m - 1; }
            next_j = (blk << 5) + stop_lane;
        }
        const bool in_range = valid && i < next_j;
        if (in_range && !cov) { win_idx[wn + rank] = i; win_anchors[wn + rank] = an; }
        if (in_range && cov) {
            keep[i] = 0;
            sfe_result r; r.score = r.score_fwd = r.score_bwd = 0; r.status = SFE_ST_SKIPPED;
            r.tstart = r.tend = tp; r.qstart = r.qend = qp; r.cigar_off = -1; r.n_ops = r.n_ops_back = 0; r.cells = 0;
            results[i] = r;
        }
        c_cov += __popc(__ballot_sync(FULL, in_range && cov));
        wn += n_unc > room ? room : n_unc;
        j = next_j;
    }
    if (lane == 0) {
        st->cursor = j; st->win_n = wn; st->nact = nact;
        if (stats) { stats->n_anchors += c_cov; stats->n_covered += c_cov; }
    }
}

// single warp; wres = results of the compact window (phase 2)
__global__ void spec_commit_kernel(SpecState *st, const sfe_anchor *win_anchors, const sfe_result *wres, const long long *win_idx,
                                   const long long *blkmin, int min_score, sfe_box *accepted, long long accepted_cap,
                                   sfe_box *act, sfe_box *local, uint8_t *keep, sfe_result *results, sfe_stats *stats)
{
    const int lane = threadIdx.x & 31;
    const long long wn = st->win_n;
    long long nacc = st->nacc, nloc = 0;
    long long c_kept = 0, c_cov = 0, c_below = 0;
    unsigned long long cells_tot = 0, cells_cov = 0;
    bool overflow = false;
    for (long long base = 0; base < wn; base += 32) {
        nloc = retire_boxes(local, nloc, blkmin[win_idx[base] >> 5], lane);
        const long long w = base + lane;
        const bool valid = w < wn;
        long long tp = 0, qp = 0, gi = 0; int strand = 0, score = 0; unsigned long long cells = 0;
        sfe_box mine; mine.tstart = mine.tend = mine.qstart = mine.qend = 0; mine.strand = 0; mine.reserved = 0;
        sfe_result r;
        if (valid) {
            gi = win_idx[w]; r = wres[w];
            tp = win_anchors[w].tpos; qp = win_anchors[w].qpos; strand = win_anchors[w].strand >= 0 ? 1 : -1;
            score = r.score; cells = r.cells;
            mine.tstart = r.tstart; mine.tend = r.tend; mine.qstart = r.qstart; mine.qend = r.qend; mine.strand = strand;
        }
        bool cov = false;
        for (long long k = 0; k < nloc; k++) { const sfe_box b = local[k]; cov = cov || box_has(b, tp, qp, strand); }
        cov = cov && valid;
        const bool live = valid && !cov, cand = live && score >= min_score;
        const unsigned kmask = decide_block(valid, live, cand, cov, mine, tp, qp, strand, lane);
        const bool kept = (kmask >> lane) & 1u;
        if (kept) {
            const long long r = __popc(kmask & ((1u << lane) - 1));
            local[nloc + r] = mine;
            if (nacc + r < accepted_cap) accepted[nacc + r] = mine;
        }
        {
            const long long nk = __popc(kmask);
            if (nacc + nk > accepted_cap) overflow = true;
            nloc += nk; nacc += nk;
        }
        __syncwarp();
        if (valid) {
            keep[gi] = cov ? 0 : (kept ? 1 : 2);
            results[gi] = r;
            c_kept += kept; c_cov += cov; c_below += (!cov && !kept);
            cells_tot += cells; if (cov) cells_cov += cells;
        }
    }
    // the boxes of this window that can still cover a later anchor join the persistent active list
    long long nact = st->nact;
    for (long long k = lane; k < nloc; k += 32) act[nact + k] = local[k];
    nact += nloc;
    for (int o = 16; o > 0; o >>= 1) {
        c_kept += __shfl_xor_sync(FULL, c_kept, o); c_cov += __shfl_xor_sync(FULL, c_cov, o);
        c_below += __shfl_xor_sync(FULL, c_below, o);
        cells_tot += __shfl_xor_sync(FULL, cells_tot, o); cells_cov += __shfl_xor_sync(FULL, cells_cov, o);
    }
    if (lane == 0) {
        st->nact = nact; st->nacc = nacc; if (overflow) st->overflow = 1;
        if (stats) {
            stats->n_anchors += wn; stats->n_kept += c_kept; stats->n_covered += c_cov; stats->n_below += c_below;
            stats->cells_total += cells_tot; stats->cells_covered += cells_cov;
            stats->n_extended += wn; stats->n_windows += 1;
        }
    }
}

__global__ void spec_finish_kernel(const SpecState *st, long long *n_accepted_io)
{
    if (threadIdx.x == 0) *n_accepted_io = st->overflow ? -st->nacc : st->nacc;
}

// SFE_CIGAR_KEPT_ONLY: the kept anchors, in anchor order, for the final traceback batch (single warp), and the scatter back.
__global__ void spec_gather_kept_kernel(const sfe_anchor *anchors, const uint8_t *keep, long long n, sfe_anchor *kept_anchors,
                                        long long *kept_idx, long long *n_kept)
{
    const int lane = threadIdx.x & 31;
    long long w = 0;
    for (long long base = 0; base < n; base += 32) {
        const long long i = base + lane;
        const bool k = i < n && keep[i] == 1;
        const unsigned m = __ballot_sync(FULL, k);
        if (k) { const long long d = w + __popc(m & ((1u << lane) - 1)); kept_anchors[d] = anchors[i]; kept_idx[d] = i; }
        w += __popc(m);
    }
    if (lane == 0) *n_kept = w;
}

__global__ void spec_scatter_kept_kernel(const sfe_result *kres, const long long *kept_idx, long long nk, sfe_result *results)
{
    const long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (k < nk) results[kept_idx[k]] = kres[k];
}

int sfe_launch_spec_gather_kept(const sfe_anchor *anchors, const uint8_t *keep, long long n, sfe_anchor *kept_anchors,
                                long long *kept_idx, long long *n_kept, cudaStream_t st)
{
    SFE_KL spec_gather_kept_kernel<<<1, 32, 0, st>>>(anchors, keep, n, kept_anchors, kept_idx, n_kept);
    SFE_LAUNCH_CHECK();
}

int sfe_launch_spec_scatter_kept(const sfe_result *kres, const long long *kept_idx, long long nk, sfe_result *results, cudaStream_t st)
{
    if (nk <= 0) return SFE_OK;
    const int bs = 256;
    SFE_KL spec_scatter_kept_kernel<<<(unsigned)((nk + bs - 1) / bs), bs, 0, st>>>(kres, kept_idx, nk, results);
    SFE_LAUNCH_CHECK();
}

int sfe_launch_spec_prepare(const sfe_anchor *anchors, long long n, long long *blkmin, void *state, const sfe_box *accepted,
                            const long long *n_accepted, sfe_box *act, cudaStream_t st)
{
    const int bs = 256;
    SFE_KL block_min_kernel<<<(unsigned)((n + bs - 1) / bs), bs, 0, st>>>(anchors, n, blkmin);
    SFE_KL suffix_min_kernel<<<1, 32, 0, st>>>(blkmin, (n + 31) >> 5);
    SFE_KL spec_init_kernel<<<1, 32, 0, st>>>((SpecState *)state, accepted, n_accepted, act);
    SFE_LAUNCH_CHECK();
}

int sfe_launch_spec_scan(void *state, const sfe_anchor *anchors, long long n, const long long *blkmin, long long K, sfe_box *act,
                         long long *win_idx, sfe_anchor *win_anchors, uint8_t *keep, sfe_result *results, sfe_stats *stats,
                         cudaStream_t st)
{
    SFE_KL spec_scan_kernel<<<1, 32, 0, st>>>((SpecState *)state, anchors, n, blkmin, K, act, win_idx, win_anchors, keep, results, stats);
    SFE_LAUNCH_CHECK();
}

int sfe_launch_spec_commit(void *state, const sfe_anchor *win_anchors, const sfe_result *wres, const long long *win_idx,
                           const long long *blkmin, int min_score, sfe_box *accepted, long long accepted_cap, sfe_box *act,
                           sfe_box *local, uint8_t *keep, sfe_result *results, sfe_stats *stats, cudaStream_t st)
{
    SFE_KL spec_commit_kernel<<<1, 32, 0, st>>>((SpecState *)state, win_anchors, wres, win_idx, blkmin, min_score, accepted, accepted_cap,
                                         act, local, keep, results, stats);
    SFE_LAUNCH_CHECK();
}

int sfe_launch_spec_finish(const void *state, long long *n_accepted_io, cudaStream_t st)
{
    SFE_KL spec_finish_kernel<<<1, 32, 0, st>>>((const SpecState *)state, n_accepted_io);
    SFE_LAUNCH_CHECK();
}
