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

__global__ void spec_gather_results_kernel(const sfe_result *results, const long long *kept_idx, long long nk, sfe_result *kres)
{
    const long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (k < nk) kres[k] = results[kept_idx[k]];
}

// one byte per anchor for sfe_launch_tickets: 1 + floor(log2(span)) of an extension that is already known
__global__ void len_bins_kernel(const sfe_result *res, long long n, uint8_t *prio)
{
    const long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (k >= n) return;
    long long span = res[k].tend - res[k].tstart;
    const long long qs = res[k].qend - res[k].qstart;
    if (qs > span) span = qs;
    if (span < 1) span = 1;
    if (span > 0x3fffffff) span = 0x3fffffff;
    prio[k] = (uint8_t)(1 + (31 - __clz((int)span)));
}

int sfe_launch_len_bins(const sfe_result *res, long long n, uint8_t *prio, cudaStream_t st)
{
    if (n <= 0) return SFE_OK;
    const int bs = 256;
    SFE_KL len_bins_kernel<<<(unsigned)((n + bs - 1) / bs), bs, 0, st>>>(res, n, prio);
    SFE_LAUNCH_CHECK();
}

// nk > 0: results[kept_idx[k]] = kres[k];  nk < 0: the other way round for -nk entries (first argument = results)
int sfe_launch_spec_scatter_kept(const sfe_result *kres, const long long *kept_idx, long long nk, sfe_result *results, cudaStream_t st)
{
    if (nk < 0) {
        const int bs = 256;
        SFE_KL spec_gather_results_kernel<<<(unsigned)((-nk + bs - 1) / bs), bs, 0, st>>>(kres, kept_idx, -nk, results);
        SFE_LAUNCH_CHECK();
    }
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

// =====================================================================================================
// Algorithm 3 with PREDICTED LEADERS (SFE_SPEC_LEADERS): the same in-order commit, a smarter phase 1.
//
// Algorithm 3 takes "the next K unmasked seeds" as its batch.  In the dense-anchor regimes the
// paper is about, almost all of those lie on the diagonal of the batch's first alignment and are thrown away in phase 3
// (shadow work) -- after each of them has cost one full-length extension.  Which anchors are speculated on
// is a free choice as long as phase 3 stays in order: an anchor may be DECIDED only when every earlier anchor is, and it
// is decided either because a kept box covers it (no extension needed: Algorithm 1 would not extend it either) or because
// its extension is available.  So:
//   classify  (parallel, once)   an anchor is a FOLLOWER if a close earlier anchor of the same strand lies on (nearly) the
//                                same diagonal with no N run in between -- it will most likely be covered by that
//                                anchor's alignment -- else a LEADER; leaders with followers right behind them are
//                                flagged long-likely (their tickets are issued first);
//   advance   (one warp)         commit from the cursor in anchor order using the results cached so far; STOP at the
//                                first anchor that is neither covered nor extended; then build the next batch: that
//                                anchor (plus a doubling number of its successors after repeated stops in one region: a
//                                mispredicted stretch costs O(log) batches) and every not yet extended leader in the
//                                look-ahead span;
//   extend    (sfe_ydrop_batch)  results are cached per anchor: nothing is ever extended twice;
// until the cursor reaches the end.  The kept set, scores, boxes and CIGARs are Algorithm 1's for ANY classification
// (tests run it with adversarial ones); the classification only decides how much is extended and how many batches it takes.
// =====================================================================================================
struct SpecLState { long long cursor, win_n, nact, nacc, overflow, spec_hi, esc, last_stop, n_forced, n_stops, n_cold, plist_rd;
                    unsigned long long plist_n; };

enum { CLS_FOLLOWER = 0, CLS_LEADER = 1, CLS_LEADER_LONG = 2, CLS_PROMOTED = 3 };

static __device__ __forceinline__ bool is_n_at(const uint8_t *nmask, long long k, long long len)
{
    return k >= 0 && k < len && ((nmask[k >> 3] >> (k & 7)) & 1);
}

// number of N among target bases [a, b)
static __device__ long long count_n(const uint8_t *nmask, long long a, long long b)
{
    long long c = 0;
    for (long long k = a; k < b;) {
        if ((k & 7) == 0 && k + 8 <= b) { c += __popc((unsigned)nmask[k >> 3]); k += 8; }
        else { c += (nmask[k >> 3] >> (k & 7)) & 1; k++; }
    }
    return c;
}

__global__ void spec_classify_kernel(const sfe_anchor *anchors, long long n, const uint8_t *t_nmask, long long t_len,
                                     const uint8_t *q_nmask, const uint8_t *qrc_nmask, long long q_len, int tol, long long gap,
                                     int lookback, int n_break, uint8_t *cls, uint8_t *lead_prio)
{
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= n) return;
    const sfe_anchor a = anchors[i];
    const int strand = a.strand >= 0 ? 1 : -1;
    const uint8_t *qm = strand > 0 ? q_nmask : qrc_nmask;
    auto dead_end = [&](const sfe_anchor &x) {              // both first diagonal cells pair with an N: both halves die at once
        const uint8_t *m = x.strand >= 0 ? q_nmask : qrc_nmask;
        if (!m) return false;
        const bool f = is_n_at(t_nmask, x.tpos, t_len) || is_n_at(m, x.qpos, q_len);
        const bool b = is_n_at(t_nmask, x.tpos - 1, t_len) || is_n_at(m, x.qpos - 1, q_len);
        return f && b;
    };
    uint8_t c = CLS_LEADER;
    // an anchor inside an N run leads (nobody covers it before it has been extended).  Its extension is usually empty -- but
    // within ydrop / |n_score| bases of the run's edge it climbs out and runs the full length of what lies beyond (measured on
    // configs[4]: the longest halves of a batch started there), so its reach is estimated like everybody's below.
    const bool inside_n = qm && dead_end(a);
    const long long diag = a.tpos - a.qpos;
    for (long long j = i - 1; !inside_n && j >= 0 && j >= i - lookback; j--) {
        const sfe_anchor p = anchors[j];
        if (a.tpos - p.tpos > gap) break;                   // anchors are in target order (any other order: everybody leads)
        if (a.tpos < p.tpos) break;
        if ((p.strand >= 0 ? 1 : -1) != strand || p.pair != a.pair) continue;
        const long long dd = (p.tpos - p.qpos) - diag;
        if (dd > tol || dd < -tol) continue;
        if (dead_end(p)) continue;
        if (count_n(t_nmask, p.tpos, a.tpos) >= n_break) break;
        c = CLS_FOLLOWER;
        break;
    }
    uint8_t pr = 0;
    if (c == CLS_LEADER) {
        // Long-likely, and how long: follow the anchors on this one's diagonal in both directions (same strand / pair, diagonal
        // within tol of the LAST one found, no gap wider than `gap`, no long N run in between) -- the reach of that chain is a
        // proxy of the alignment's span, which nothing else knows before the extension has run.  Forward it is the anchors that
        // would follow this one; backward it is ground an earlier leader is expected to cover, but this anchor's LEFT half runs
        // over it all the same when that leader's extension stopped short of it (measured on configs[4]: the longest halves
        // of a batch were such left halves).  The log2 of the longer reach is the priority of both tickets (longest first).
        // (Priority only: an N run shorter than n_cross can be bridged by two gaps within ydrop, so it does not end the reach;
        // N bases add up over consecutive hops until a hop has none.)
        const int n_cross = 2 * n_break + n_break / 2;
        long long span = 0; int nf = 0;
#pragma unroll 1
        for (int dir = 1; dir >= -1; dir -= 2) {
            long long last_t = a.tpos, last_d = diag, n_acc = 0;                 // n_acc: N bases since the last hop without any
            for (long long j = i + dir; j >= 0 && j < n && j <= i + (1 << 17) && j >= i - (1 << 17); j += dir) {
                const sfe_anchor p = anchors[j];
                const long long dt = dir > 0 ? p.tpos - last_t : last_t - p.tpos;
                if (dt > gap || (dir > 0 ? p.tpos < a.tpos : p.tpos > a.tpos)) break;
                if ((p.strand >= 0 ? 1 : -1) != strand || p.pair != a.pair) continue;
                const long long dd = (p.tpos - p.qpos) - last_d;
                if (dd <= tol && dd >= -tol) {
                    const long long cn = count_n(t_nmask, dir > 0 ? last_t : p.tpos, dir > 0 ? p.tpos : last_t);
                    n_acc = cn ? n_acc + cn : 0;
                    if (n_acc >= n_cross) break;
                    last_t = p.tpos; last_d = p.tpos - p.qpos; nf++;
                }
            }
            const long long sp = (dir > 0 ? last_t - a.tpos : a.tpos - last_t) + 1;
            if (sp > span) span = sp;
        }
        if (nf > 0) {
            c = CLS_LEADER_LONG;
            if (span > 0x3fffffff) span = 0x3fffffff;
            pr = (uint8_t)(1 + (31 - __clz((int)span)));
        }
    }
    lead_prio[i] = pr;
    cls[i] = c;
}

__global__ void specl_init_kernel(SpecLState *st, const sfe_box *accepted, const long long *n_accepted, sfe_box *act)
{
    const int lane = threadIdx.x & 31;
    const long long nacc = *n_accepted;
    for (long long k = lane; k < nacc; k += 32) act[k] = accepted[k];
    if (lane == 0) { st->cursor = 0; st->win_n = 0; st->nact = nacc; st->nacc = nacc; st->overflow = 0; st->spec_hi = 0; st->esc = 1;
                     st->last_stop = -1; st->n_forced = 0; st->n_stops = 0; st->n_cold = 0; st->plist_rd = 0; st->plist_n = 0ULL; }
}

// ext_state[i]: 0 = not extended, 1 = extended (results[i] holds it), 2 = queued in the batch being built
// single warp
__global__ void spec_advance_kernel(SpecLState *st, const sfe_anchor *anchors, long long n, const long long *blkmin, long long K,
                                    long long span, int esc_max, int tol, long long gap, int lookback, const uint8_t *cls, uint8_t *ext_state, sfe_box *act,
                                    int min_score, sfe_box *accepted, long long accepted_cap, long long *win_idx,
                                    sfe_anchor *win_anchors, uint8_t *win_prio, uint8_t *keep, sfe_result *results, sfe_stats *stats,
                                    const int32_t *plist, const uint8_t *lead_prio)
{
    const int lane = threadIdx.x & 31;
    long long j = st->cursor, nact = st->nact, nacc = st->nacc;
    long long c_kept = 0, c_cov = 0, c_below = 0, c_dec = 0;
    unsigned long long cells_tot = 0, cells_cov = 0;
    bool overflow = false, stopped = false;
    // ---- phase 3, in order, as far as the cached extensions reach ----
    while (j < n && !stopped) {
        const long long blk = j >> 5;
        nact = retire_boxes(act, nact, blkmin[blk], lane);
        const long long i = (blk << 5) + lane;
        const bool valid = i >= j && i < n;
        long long tp = 0, qp = 0; int strand = 0, score = 0; unsigned long long cells = 0; bool ext = false;
        sfe_box mine; mine.tstart = mine.tend = mine.qstart = mine.qend = 0; mine.strand = 0; mine.reserved = 0;
        if (valid) {
            const sfe_anchor an = anchors[i];
            tp = an.tpos; qp = an.qpos; strand = an.strand >= 0 ? 1 : -1;
            ext = ext_state[i] == 1;
            if (ext) {
                const sfe_result r = results[i];
                score = r.score; cells = r.cells;
                mine.tstart = r.tstart; mine.tend = r.tend; mine.qstart = r.qstart; mine.qend = r.qend; mine.strand = strand;
            }
        }
        bool cov = false;
        for (long long k = 0; k < nact; k++) { const sfe_box b = act[k]; cov = cov || box_has(b, tp, qp, strand); }
        cov = cov && valid;
        const bool live = valid && !cov, cand = live && ext && score >= min_score;
        const unsigned kmask_all = decide_block(valid, live, cand, cov, mine, tp, qp, strand, lane);
        // the first anchor that is neither covered nor extended cannot be decided: everything from there on waits
        const unsigned stopm = __ballot_sync(FULL, valid && !cov && !ext);
        const int stop_lane = stopm ? __ffs(stopm) - 1 : 32;
        const unsigned below_stop = stop_lane >= 32 ? 0xffffffffu : ((1u << stop_lane) - 1u);
        const unsigned kmask = kmask_all & below_stop;
        const bool decided = valid && lane < stop_lane;
        const bool kept = (kmask >> lane) & 1u;
        if (kept) {
            const long long r = __popc(kmask & ((1u << lane) - 1));
            act[nact + r] = mine;
            if (nacc + r < accepted_cap) accepted[nacc + r] = mine;
        }
        {
            const long long nk = __popc(kmask);
            if (nacc + nk > accepted_cap) overflow = true;
            nact += nk; nacc += nk;
        }
        __syncwarp();
        if (decided) {
            keep[i] = cov ? 0 : (kept ? 1 : 2);
            if (!ext) {                                       // covered before anybody extended it: as in Algorithm 1
                sfe_result r; r.score = r.score_fwd = r.score_bwd = 0; r.status = SFE_ST_SKIPPED;
                r.tstart = r.tend = tp; r.qstart = r.qend = qp; r.cigar_off = -1; r.n_ops = r.n_ops_back = 0; r.cells = 0;
                results[i] = r;
            }
            c_dec++; c_kept += kept; c_cov += cov; c_below += (!cov && !kept);
            cells_tot += cells; if (cov) cells_cov += cells;
        }
        stopped = stop_lane < 32;
        j = stopped ? (blk << 5) + stop_lane : (((blk + 1) << 5) < n ? ((blk + 1) << 5) : n);
    }
    // ---- the next batch: the anchor(s) the commit waits for, then every leader of the look-ahead span ----
    long long esc = st->esc, last_stop = st->last_stop, n_forced = 0;
    bool cold = false; long long cdiag = 0; int cstrand = 0;
    if (stopped) {
        esc = (last_stop >= 0 && j - last_stop <= 4096) ? (2 * esc < esc_max ? 2 * esc : esc_max) : 1;
        last_stop = j;
        // Cold diagonal: the nearest EXTENDED predecessor on the stop anchor's diagonal came out below tau (it masks
        // nothing, R18), so the anchors behind it on that diagonal are not covered either and will most likely score the
        // same: false homology, repeats, a diagonal through N runs.  Their extensions are short and independent of one
        // another -- take every one of them in the look-ahead at once instead of one commit stop each.
        const sfe_anchor sa = anchors[j];
        cdiag = sa.tpos - sa.qpos; cstrand = sa.strand >= 0 ? 1 : -1;
        long long best_d = 0x7fffffffffffffffLL; int best_below = 0;
        for (long long base = j - 1; base >= 0 && base > j - 1 - lookback; base -= 32) {
            const long long x = base - lane;
            long long d = 0x7fffffffffffffffLL; int below = 0;
            if (x >= 0 && x > j - 1 - lookback && ext_state[x] == 1) {
                const sfe_anchor pa = anchors[x];
                const long long dd = (pa.tpos - pa.qpos) - cdiag;
                if ((pa.strand >= 0 ? 1 : -1) == cstrand && pa.pair == sa.pair && dd <= tol && dd >= -tol && sa.tpos - pa.tpos <= gap && sa.tpos >= pa.tpos) {
                    d = j - x; below = results[x].score < min_score;
                }
            }
            for (int o = 16; o > 0; o >>= 1) {
                const long long od = __shfl_xor_sync(FULL, d, o); const int ob = __shfl_xor_sync(FULL, below, o);
                if (od < d) { d = od; below = ob; }
            }
            if (d < best_d) { best_d = d; best_below = below; }
        }
        cold = esc_max > 1 && best_d != 0x7fffffffffffffffLL && best_below;      // esc_max == 1: no escalation of any kind
    }
    long long wn = 0;
    if (j < n) {
        // forced: the first `esc` not-extended anchors from the cursor that no active box covers -- or, on a cold diagonal,
        // every not-extended anchor of that diagonal in the next 8192
        long long want = stopped ? (cold ? K : esc) : 0;
        for (long long p = j; p < n && want > 0 && wn < K && p < j + 8192; ) {
            const long long blk = p >> 5;
            const long long i = (blk << 5) + lane;
            const bool valid = i >= p && i < n;
            sfe_anchor an; an.tpos = an.qpos = 0; an.pair = 0; an.strand = 1;
            bool take = false;
            if (valid) {
                an = anchors[i];
                take = ext_state[i] == 0;
                if (cold) {
                    const long long dd = (an.tpos - an.qpos) - cdiag;
                    take = take && (an.strand >= 0 ? 1 : -1) == cstrand && dd <= 2 * tol && dd >= -2 * tol;
                }
            }
            bool cov = false;
            const int strand = an.strand >= 0 ? 1 : -1;
            for (long long k = 0; k < nact; k++) { const sfe_box b = act[k]; cov = cov || box_has(b, an.tpos, an.qpos, strand); }
            take = take && !cov;
            unsigned m = __ballot_sync(FULL, take);
            const long long room = (want < K - wn) ? want : (K - wn);
            while ((long long)__popc(m) > room) m &= ~(0x80000000u >> __clz(m));     // drop the highest lanes
            if ((m >> lane) & 1u) {
                const long long d = wn + __popc(m & ((1u << lane) - 1));
                win_idx[d] = i; win_anchors[d] = an; win_prio[d] = cold ? 0 : 1; ext_state[i] = 2;
            }
            const long long got = __popc(m);
            wn += got; want -= got; n_forced += got;
            p = ((blk + 1) << 5);
        }
        // promoted followers (spec_promote_kernel's list; any order): those still ahead of the cursor and not extended yet
        {
            long long rd = st->plist_rd;
            const long long pn = (long long)st->plist_n;
            while (rd < pn && wn < K) {
                const long long x = rd + lane;
                long long i = -1;
                sfe_anchor an; an.tpos = an.qpos = 0; an.pair = 0; an.strand = 1;
                bool take = false;
                if (x < pn) {
                    i = plist[x];
                    if (i >= j && i < j + span && ext_state[i] == 0) { an = anchors[i]; take = true; }
                }
                if (__any_sync(FULL, take)) {
                    bool cov = false;
                    const int strand = an.strand >= 0 ? 1 : -1;
                    for (long long k = 0; k < nact; k++) { const sfe_box b = act[k]; cov = cov || box_has(b, an.tpos, an.qpos, strand); }
                    take = take && !cov;
                }
                unsigned m = __ballot_sync(FULL, take);
                long long adv = 32;
                if ((long long)__popc(m) > K - wn) {               // the batch is full: stop inside this group of 32
                    unsigned keepm = 0; long long room = K - wn;
                    for (unsigned mm = m; mm && room > 0; mm &= mm - 1, room--) keepm |= mm & (0u - mm);
                    adv = 31 - __clz(keepm) + 1;
                    m = keepm;
                }
                if ((m >> lane) & 1u) {
                    const long long d = wn + __popc(m & ((1u << lane) - 1));
                    win_idx[d] = i; win_anchors[d] = an; win_prio[d] = 0; ext_state[i] = 2;
                }
                wn += __popc(m);
                rd += adv;
            }
            if (rd > pn) rd = pn;
            if (lane == 0) st->plist_rd = rd;
        }
        // speculative: leaders of [max(spec_hi, cursor), cursor + span) that are not extended yet
        long long p = st->spec_hi > j ? st->spec_hi : j;
        const long long hi = (j + span < n) ? j + span : n;
        while (p < hi && wn < K) {
            const long long blk = p >> 5;
            const long long i = (blk << 5) + lane;
            const bool valid = i >= p && i < hi;
            sfe_anchor an; an.tpos = an.qpos = 0; an.pair = 0; an.strand = 1;
            bool take = false; uint8_t c = 0;
            if (valid) {
                c = cls[i];
                if (c != CLS_FOLLOWER && ext_state[i] == 0) { an = anchors[i]; take = true; }
            }
            if (__any_sync(FULL, take)) {
                bool cov = false;
                const int strand = an.strand >= 0 ? 1 : -1;
                for (long long k = 0; k < nact; k++) { const sfe_box b = act[k]; cov = cov || box_has(b, an.tpos, an.qpos, strand); }
                take = take && !cov;
            }
            unsigned m = __ballot_sync(FULL, take);
            long long next_p = ((blk + 1) << 5) < hi ? ((blk + 1) << 5) : hi;
            if ((long long)__popc(m) > K - wn) {                  // the batch is full: stop inside this block
                unsigned keepm = 0; long long room = K - wn;
                for (unsigned mm = m; mm && room > 0; mm &= mm - 1, room--) keepm |= mm & (0u - mm);
                const int last = 31 - __clz(keepm);
                next_p = (blk << 5) + last + 1;
                m = keepm;
            }
            if ((m >> lane) & 1u) {
                const long long d = wn + __popc(m & ((1u << lane) - 1));
                win_idx[d] = i; win_anchors[d] = an; win_prio[d] = c == CLS_LEADER_LONG ? lead_prio[i] : 0; ext_state[i] = 2;
            }
            wn += __popc(m);
            p = next_p;
        }
        if (lane == 0) st->spec_hi = p;
    }
    for (int o = 16; o > 0; o >>= 1) {
        c_kept += __shfl_xor_sync(FULL, c_kept, o); c_cov += __shfl_xor_sync(FULL, c_cov, o);
        c_below += __shfl_xor_sync(FULL, c_below, o); c_dec += __shfl_xor_sync(FULL, c_dec, o);
        cells_tot += __shfl_xor_sync(FULL, cells_tot, o); cells_cov += __shfl_xor_sync(FULL, cells_cov, o);
    }
    if (lane == 0) {
        st->cursor = j; st->win_n = wn; st->nact = nact; st->nacc = nacc; if (overflow) st->overflow = 1;
        st->esc = esc; st->last_stop = last_stop; st->n_forced += n_forced; st->n_stops += stopped ? 1 : 0; st->n_cold += cold ? 1 : 0;
        if (stats) {
            stats->n_anchors += c_dec; stats->n_kept += c_kept; stats->n_covered += c_cov; stats->n_below += c_below;
            stats->cells_total += cells_tot; stats->cells_covered += cells_cov;
            stats->n_extended += wn; if (wn > 0) stats->n_windows += 1;
        }
    }
}

// cache the batch's results per anchor (anchor order) and mark them extended
__global__ void spec_store_kernel(const sfe_result *wres, const long long *win_idx, long long wn, sfe_result *results, uint8_t *ext_state)
{
    const long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (k >= wn) return;
    const long long i = win_idx[k];
    results[i] = wres[k];
    ext_state[i] = 1;
}

// After a batch: anchors the classifier called followers are promoted to leaders where the result of the anchor they
// follow shows that they will NOT be covered by it -- it scored below tau (R18: it masks nothing; a cold diagonal), or
// they lie beyond its box (an alignment that stopped right at its own anchor, e.g. at the edge of an N run: every later
// anchor of that diagonal starts another one).  They are extended together in the next batch instead of costing one
// commit stop each.  Parallel over the batch; scans ahead while the target distance is within `reach`.
__global__ void spec_promote_kernel(const sfe_result *wres, const long long *win_idx, long long wn, const sfe_anchor *anchors,
                                    long long n, int min_score, int tol, long long reach, int max_ahead, const uint8_t *ext_state,
                                    uint8_t *cls, SpecLState *st, int32_t *plist)
{
    const long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (k >= wn) return;
    const long long i = win_idx[k];
    const sfe_result r = wres[k];
    const sfe_anchor a = anchors[i];
    const bool below = r.score < min_score;
    const long long diag = a.tpos - a.qpos;
    const int strand = a.strand >= 0 ? 1 : -1;
    for (long long j = i + 1; j < n && j <= i + max_ahead; j++) {
        const sfe_anchor f = anchors[j];
        if (f.tpos - a.tpos > reach || f.tpos < a.tpos) break;
        if ((f.strand >= 0 ? 1 : -1) != strand || f.pair != a.pair) continue;
        const long long dd = (f.tpos - f.qpos) - diag;
        if (dd > 2 * tol || dd < -2 * tol) continue;
        const uint8_t cj = cls[j];
        // the next leader / extended anchor of this diagonal owns whatever follows it
        if (cj == CLS_LEADER || cj == CLS_LEADER_LONG || ext_state[j] != 0) break;
        if (cj == CLS_PROMOTED) continue;
        if (below || f.tpos > r.tend || f.qpos > r.qend || f.tpos < r.tstart || f.qpos < r.qstart) {
            // claim the byte (FOLLOWER = 0 -> PROMOTED = 3) in its 32-bit word; the first claimer appends the anchor to the list
            const unsigned sh = 8u * (unsigned)(j & 3);
            const unsigned old = atomicOr((unsigned *)(cls + (j & ~3LL)), (unsigned)CLS_PROMOTED << sh);
            if (((old >> sh) & 0xffu) == CLS_FOLLOWER) plist[atomicAdd(&st->plist_n, 1ULL)] = (int32_t)j;
        }
    }
}

__global__ void specl_finish_kernel(const SpecLState *st, long long *n_accepted_io)
{
    if (threadIdx.x == 0) *n_accepted_io = st->overflow ? -st->nacc : st->nacc;
}

int sfe_launch_specl_prepare(const sfe_anchor *anchors, long long n, const uint8_t *t_nmask, long long t_len, const uint8_t *q_nmask,
                             const uint8_t *qrc_nmask, long long q_len, int tol, long long gap, int lookback, int n_break,
                             uint8_t *cls, uint8_t *lead_prio, uint8_t *ext_state, long long *blkmin, void *state, const sfe_box *accepted,
                             const long long *n_accepted, sfe_box *act, cudaStream_t st)
{
    const int bs = 256;
    const unsigned nb = (unsigned)((n + bs - 1) / bs);
    SFE_KL block_min_kernel<<<nb, bs, 0, st>>>(anchors, n, blkmin);
    SFE_KL suffix_min_kernel<<<1, 32, 0, st>>>(blkmin, (n + 31) >> 5);
    SFE_KL spec_classify_kernel<<<nb, bs, 0, st>>>(anchors, n, t_nmask, t_len, q_nmask, qrc_nmask, q_len, tol, gap, lookback, n_break, cls, lead_prio);
    if (cudaMemsetAsync(ext_state, 0, (size_t)n, st) != cudaSuccess) return SFE_ECUDA;
    SFE_KL specl_init_kernel<<<1, 32, 0, st>>>((SpecLState *)state, accepted, n_accepted, act);
    SFE_LAUNCH_CHECK();
}

int sfe_launch_spec_advance(void *state, const sfe_anchor *anchors, long long n, const long long *blkmin, long long K, long long span,
                            int esc_max, int tol, long long gap, int lookback, const uint8_t *cls, uint8_t *ext_state, sfe_box *act, int min_score, sfe_box *accepted,
                            long long accepted_cap, long long *win_idx, sfe_anchor *win_anchors, uint8_t *win_prio, uint8_t *keep,
                            sfe_result *results, sfe_stats *stats, const int32_t *plist, const uint8_t *lead_prio, cudaStream_t st)
{
    SFE_KL spec_advance_kernel<<<1, 32, 0, st>>>((SpecLState *)state, anchors, n, blkmin, K, span, esc_max, tol, gap, lookback, cls, ext_state, act, min_score,
                                                 accepted, accepted_cap, win_idx, win_anchors, win_prio, keep, results, stats, plist, lead_prio);
    SFE_LAUNCH_CHECK();
}

int sfe_launch_spec_store(const sfe_result *wres, const long long *win_idx, long long wn, sfe_result *results, uint8_t *ext_state,
                          cudaStream_t st)
{
    if (wn <= 0) return SFE_OK;
    const int bs = 256;
    SFE_KL spec_store_kernel<<<(unsigned)((wn + bs - 1) / bs), bs, 0, st>>>(wres, win_idx, wn, results, ext_state);
    SFE_LAUNCH_CHECK();
}

int sfe_launch_spec_promote(const sfe_result *wres, const long long *win_idx, long long wn, const sfe_anchor *anchors, long long n,
                            int min_score, int tol, long long reach, int max_ahead, const uint8_t *ext_state, uint8_t *cls, void *state,
                            int32_t *plist, cudaStream_t st)
{
    if (wn <= 0) return SFE_OK;
    const int bs = 128;
    SFE_KL spec_promote_kernel<<<(unsigned)((wn + bs - 1) / bs), bs, 0, st>>>(wres, win_idx, wn, anchors, n, min_score, tol, reach, max_ahead, ext_state, cls,
                                                                              (SpecLState *)state, plist);
    SFE_LAUNCH_CHECK();
}

int sfe_launch_specl_finish(const void *state, long long *n_accepted_io, cudaStream_t st)
{
    SFE_KL specl_finish_kernel<<<1, 32, 0, st>>>((const SpecLState *)state, n_accepted_io);
    SFE_LAUNCH_CHECK();
}
