// ydrop_block_kernel.cu -- cooperative warps per anchor-half ("8 warps per
// anchor-half ... kernel wall time / 3.3") for the LONG halves, bit-exact with the warp-systolic kernel.
//
// Why.  With the row-lagged threshold (R4, Lambda = 32) only 32 rows of one extension can be in flight, which
// is exactly one warp's wavefront: a half of n rows is a chain of ~ (n/32)(W+62) dependent warp steps
// (~140 cycles each) whatever else the GPU does, and the longest halves decide the kernel
// time (C4) or the whole run (C3, C5).  The parallelism that is left is ALONG a row.  So: one CTA per half,
// one thread per column of the live window (1024 columns), rows strictly in order:
//   M, E, H~ = max(M, E)            elementwise from the previous row (registers; the diagonal value comes from
//                                   the left neighbour by shuffle, across warps through shared memory);
//   F(i,j) = max_{j'<j} (H~(i,j') - O - X (j - j'))     one block-wide prefix maximum of a_p = H~ - O + X p
//                                   (warp scan + warp totals in shared memory + one CREDUX per warp);
//   H = max(H~, F), alive = H >= T(i), T(i) = best(rows <= i - 32) - ydrop from a ring of cumulative row bests;
//   row bounds / row best by CREDUX per warp + shared memory.
// Two __syncthreads per row, ~15 dependent shuffle levels: a row costs a few hundred cycles instead of the
// ~16 dependent wavefront steps (~2,200 cycles) of the systolic schedule.
// Exactness: E depends only on the column above, F = prefix maximum over H~ equals the recurrence over H because
// a gap opened from an H that came from F never beats extending that F (O >= 0), and by the R6 lemma cells that
// are dead (or outside the window, which starts at the first alive column of the previous row) contribute
// nothing an alive cell, its H or a pointer on an alive path depends on.  So score, end cell (first maximum,
// R7), cell count (R28) and CIGAR (R11, R12) are those of the oracle at Lambda = 32 -- same tests as ydrop_kernel.
//
// Traceback: per row one record in a backward-traversable log (64-KiB chunks of the same recycled arena):
//   4 bit-plane words per warp that lies between the first and the last alive column (plane k = __ballot of
//   pointer bit k: no packing arithmetic), then the tail {first column stored, number of words}.
// The walk (warp 0, after the DP) copies ~4096 log words at a time into shared memory, indexes the rows in
// them, and then advances up to 32 path cells per ballot exactly as walk_traceback does.
#include "ydrop_common.cuh"

#define BK_THREADS 256
#define BK_WARPS 8
#define BK_CPT 4                         // columns per thread
#define BK_WIN 1024                      // columns of the live window = BK_THREADS * BK_CPT
#define BK_WALK_WORDS 4096               // log words staged in shared memory by the walk
#define BK_DIR 64                        // rows indexed per staged window
#define BK_CHUNK_WORDS (SFE_CHUNK_BYTES / 4)
#define BK_REC_MAX (4 * 32 + 2)          // largest row record (words)
#define BK_NINF (-(1 << 30) - (1 << 29)) // identity of the prefix maximum

struct BkShared {
    int tot2[32];                        // by window rank: warp maximum of H (Lambda = 0: running best inside the row)
    int tot[32], tex[32], tht[32];       // by window rank: warp total of a (inclusive), lane 31's exclusive prefix, lane 31's H~
    int edge[32];                        // by warp id: gated H - OX of lane 31 after the row (next row's diagonal)
    int wmax[32], wcol[32], wL[32], wR[32];
    int cum[64];                         // cumulative best over alive cells through row r, ring indexed r & 63
    int best, best_i, best_j;            // first maximum so far (warp 0)
    int best_chunk, best_wpos;           // log position just after the best row's record
    int new_chunk;                       // chunk popped by warp 0 for everybody
    int dir_base[BK_DIR], dir_c0[BK_DIR], dir_nw[BK_DIR];
    uint32_t walk[BK_WALK_WORDS];
    uint32_t opsbuf[SFE_WALK_OPS];
};

// inclusive prefix maximum over the warp
static __device__ __forceinline__ int warp_scan_max(int v, int lane)
{
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(FULL, v, o); if (lane >= o) v = max(v, y); }
    return v;
}

// Walk the row log from the end cell to the origin (warp 0; every lane holds the same state).  The record of row
// `top` ends at word `wend` of `chunk`.  Returns false if the origin was not reached (internal error guard).
static __device__ bool block_walk(const YdParams &p, BkShared &sh, const int end_i, const int end_j, int chunk, int wend,
                                  const int lane, uint32_t &ops_seg, int &n_ops, bool &ops_ok)
{
    OpsWriter ow;
    ow.buf = sh.opsbuf; ow.stage = p.ops_stage; ow.used = &p.counters[CNT_OPS]; ow.cap = p.ops_cap;
    ow.nbuf = 0; ow.nops = 0; ow.cur_op = -1; ow.run = 0; ow.prev_seg = SFE_NO_SEG; ow.ok = true;
    ops_seg = SFE_NO_SEG; n_ops = 0; ops_ok = true;
    if (end_i == 0 && end_j == 0) return true;
    if (chunk < 0) return false;
    int i = end_i, j = end_j, state = 0;
    int top = end_i, ndir = 0, base0 = 0;                  // rows top, top-1, .., top-ndir+1 are indexed; walk[0] = chunk word base0
    long long guard = 3LL * ((long long)end_i + end_j) + 64;
    while (!(i == 0 && j == 0 && state == 0)) {
        if (--guard < 0) return false;
        if (top - i >= ndir) {                            // row i is below the indexed rows: stage the words before them
            if (ndir > 0) { wend = sh.dir_base[ndir - 1]; top -= ndir; }
            if (wend <= 1) {                              // this chunk is used up: the log continues in the previous one
                chunk = __ldcg(p.chunk_prev + chunk);
                if (chunk < 0) return false;
                wend = (int)__ldcg(p.pool + (size_t)chunk * BK_CHUNK_WORDS);
            }
            const int lo = max(1, wend - BK_WALK_WORDS);
            __syncwarp();
            const uint32_t *src = p.pool + (size_t)chunk * BK_CHUNK_WORDS;
            for (int x = lo + lane; x < wend; x += 32) sh.walk[x - lo] = __ldcg(src + x);
            base0 = lo;
            __syncwarp();
            int k = 0;
            if (lane == 0) {                              // index the records, last one first
                int e = wend;
                while (k < BK_DIR && e - 2 >= lo) {
                    const int nw = (int)sh.walk[e - 1 - lo], c0 = (int)sh.walk[e - 2 - lo];
                    const int start = e - 2 - nw;
                    if (nw < 16 || nw > 128 || start < lo) break;
                    sh.dir_base[k] = start; sh.dir_c0[k] = c0; sh.dir_nw[k] = nw;
                    e = start; k++;
                }
            }
            ndir = __shfl_sync(FULL, k, 0);
            __syncwarp();
            if (ndir == 0 || top != i) return false;
        }
        // lane x examines the x-th cell from (i, j) in the direction of the current state
        const int di = state == 2 ? 0 : 1, dj = state == 1 ? 0 : 1;
        const int ix = i - lane * di, jx = j - lane * dj;
        const int k = top - ix;
        bool valid = ix >= 0 && jx >= 0 && k < ndir;
        uint32_t nib = 0;
        if (valid) {
            const int pos = jx - sh.dir_c0[k];
            valid = pos >= 0 && pos < 8 * sh.dir_nw[k];
            if (valid) {
                nib = (sh.walk[(sh.dir_base[k] - base0) + (pos >> 3)] >> (16 * ((pos >> 2) & 1) + 4 * (3 - (pos & 3)))) & 15u;
            }
        }
        // nib: bit3 = H not from M, bit2 = H not from E, bit1 = E extended, bit0 = F extended (R11)
        const bool cont = state == 0 ? !(nib & 8u) : (state == 1 ? (nib & 2u) != 0 : (nib & 1u) != 0);
        const bool origin = ix == 0 && jx == 0;
        const uint32_t stop = __ballot_sync(FULL, !(valid && cont) || origin);
        const uint32_t vmask = __ballot_sync(FULL, valid);
        const int pstop = stop ? __ffs(stop) - 1 : 32;
        const bool stop_valid = pstop < 32 && ((vmask >> pstop) & 1u);
        if (pstop == 0 && !stop_valid && top - i < ndir) return false;      // the current cell itself is not in its record
        if (state == 0) {
            ow.emit(SFE_OP_M, pstop, lane);
            i -= pstop; j -= pstop;
            if (stop_valid && !(i == 0 && j == 0)) {
                const uint32_t nb = __shfl_sync(FULL, nib, pstop);
                state = (nb & 4u) ? 2 : 1;
            }
        } else if (state == 1) {
            const int cnt = stop_valid ? pstop + 1 : pstop;
            ow.emit(SFE_OP_I, cnt, lane);
            i -= cnt;
            if (stop_valid) state = 0;
        } else {
            const int cnt = stop_valid ? pstop + 1 : pstop;
            ow.emit(SFE_OP_D, cnt, lane);
            j -= cnt;
            if (stop_valid) state = 0;
        }
    }
    if (ow.cur_op >= 0) ow.push(lane);
    ow.flush(lane);
    ops_seg = ow.prev_seg; n_ops = ow.nops; ops_ok = ow.ok;
    return true;
}

template <bool TB, bool LAG0>
static __device__ void block_half(const YdParams &p, const int hid, BkShared &sh)
{
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    sfe_half out;
    out.score = 0; out.end_i = 0; out.end_j = 0; out.status = 0; out.cells = 0;
    out.ops_seg = SFE_NO_SEG; out.n_ops = 0; out.n_strips = 0; out.n_rec = 0; out.steps = 0; out.max_steps = 0;
    out.cycles = 0; out.smid = 0; out.wslot = 0;
    const long long clk0 = clock64();
    HalfGeom g;
    if (!half_setup(p, hid, g)) {
        out.status = SFE_ST_BAD_ANCHOR;
        if (tid == 0) p.halves[hid] = out;
        return;
    }
    const int OX = p.OX, X = p.X;
    const uint32_t srow_hi = p.srow_hi;

    // ---- row-log writer state (block-uniform copies in every thread) ----
    int cur_chunk = -1, wpos = BK_CHUNK_WORDS;            // wpos: next free word of the current chunk (word 0 = used words)
    bool tb_ok = TB;
    long long n_words = 0;

    if (tid < 64) sh.cum[tid] = 0;
    if (tid == 0) { sh.best = 0; sh.best_i = 0; sh.best_j = 0; sh.best_chunk = -1; sh.best_wpos = 0; }
    if (tid < BK_WARPS) sh.edge[tid] = SFE_NEG;
    __syncthreads();

    int ws = 0, ws_prev = 0;                              // window start of this / the previous row (multiples of 128)
    int myc0 = -1;                                        // first of my BK_CPT columns
    int Hu[BK_CPT], Eu[BK_CPT];                           // previous-row state of my columns: gated H - OX, E
    uint32_t sel[BK_CPT];
#pragma unroll
    for (int k = 0; k < BK_CPT; k++) { Hu[k] = SFE_NEG; Eu[k] = SFE_NEG; sel[k] = 0x8880u; }
    unsigned long long cells = 0;
    int rows_done = 0, max_width = 0;
    bool wide = false, limit = false;
    uint32_t srow32 = 0u;                                 // lane l: packed scores of query row (i & ~31) + l (row 0: all 0, R8)

    for (int i = 0; i <= g.n; i++) {
        if ((i & 31) == 0) {                              // one load per lane per 32 rows instead of one per thread per row
            const int r = i + lane;
            srow32 = (r == 0 || r > g.n) ? 0u : p.srow[sfe_base(g.qc, g.qm, g.q0 + (long long)g.d * r)];
        }
        const uint32_t srow_lo = __shfl_sync(FULL, srow32, i & 31);
        if (i >= 32 && sh.cum[(i - 32) & 63] >= SFE_SCORE_LIMIT) { limit = true; break; }    // R25 (block-uniform: one shared word)
        const int T = p.ydrop_inf ? SFE_T_INF : (i >= 32 ? sh.cum[(i - 32) & 63] : 0) - p.Y;    // R4, Lambda = 32
        // ---- my columns in this row's window ----
        const int q = ((tid * BK_CPT) - ws) & (BK_WIN - 1);       // window position of my first column
        const int c0 = ws + q;
        if (c0 != myc0) {
            myc0 = c0;
#pragma unroll
            for (int k = 0; k < BK_CPT; k++) { Hu[k] = SFE_NEG; Eu[k] = SFE_NEG; sel[k] = col_selector(g, c0 + k); }
        }
        const int rank = (warp - (ws >> 7)) & (BK_WARPS - 1);     // my warp's position in the window
        // ---- diagonal of my first column: the left neighbour's previous-row value ----
        int Hd0 = __shfl_up_sync(FULL, Hu[BK_CPT - 1], 1);
        if (lane == 0) Hd0 = (c0 - 1 - ws_prev < BK_WIN) ? sh.edge[(warp - 1) & (BK_WARPS - 1)] : SFE_NEG;
        if (q == 0) Hd0 = SFE_NEG;
        if (i == 0 && c0 == 0) Hd0 = -OX;                 // the origin
        int M[BK_CPT], E[BK_CPT], Ht[BK_CPT], pa[BK_CPT];
#pragma unroll
        for (int k = 0; k < BK_CPT; k++) {
            const int Hd = k == 0 ? Hd0 : Hu[k - 1];
            const int s = prmt_sx(srow_lo, srow_hi, sel[k]);
            M[k] = Hd + s + OX;
            E[k] = __viaddmax_s32(Eu[k], -X, Hu[k]);
            Ht[k] = max(M[k], E[k]);                      // (columns beyond m: overridden on H below; their H~ only feeds columns further right)
            const int a = Ht[k] - OX + X * (q + k + 1);   // a_p = H~ - O + X p
            pa[k] = k == 0 ? a : max(pa[k - 1], a);
        }
        // ---- F: block-wide exclusive prefix maximum ----
        const int incl = warp_scan_max(pa[BK_CPT - 1], lane);
        int excl = __shfl_up_sync(FULL, incl, 1);
        if (lane == 0) excl = BK_NINF;
        const int my_tex = max(excl, pa[BK_CPT - 2]);     // what my last column sees from inside the warp
        int lHt = __shfl_up_sync(FULL, Ht[BK_CPT - 1], 1);
        const int lpre_in = __shfl_up_sync(FULL, my_tex, 1);
        if (lane == 31) { sh.tot[rank] = incl; sh.tex[rank] = my_tex; sh.tht[rank] = Ht[BK_CPT - 1]; }
        __syncthreads();                                                                      // B1
        const int t_l = lane < BK_WARPS ? sh.tot[lane] : BK_NINF;
        const int carry_prev = __reduce_max_sync(FULL, lane < rank - 1 ? t_l : BK_NINF);      // ranks < rank - 1
        const int carry = rank > 0 ? max(carry_prev, sh.tot[rank - 1]) : BK_NINF;             // ranks < rank
        const int pre0 = max(excl, carry);
        // final H of the column left of my first one (for "F extended", R11)
        int lpre = max(lpre_in, carry);
        if (lane == 0 && rank > 0) { lHt = sh.tht[rank - 1]; lpre = max(sh.tex[rank - 1], carry_prev); }
        int Hprev = q == 0 ? SFE_NEG : max(lHt, lpre - X * (q - 1));   // (q == 1: lpre = BK_NINF)
        uint32_t nibs = 0;
        int hmax = SFE_NEG, hcol = 0x7fffffff, cl = 0x7fffffff, cr = -1;
        int Hc[BK_CPT], ph[BK_CPT];
#pragma unroll
        for (int k = 0; k < BK_CPT; k++) {
            const int pk = q + k;
            const int pre = k == 0 ? pre0 : max(pre0, pa[k - 1]);
            const int F = pre - X * pk;                   // window position 0: pre = BK_NINF (nothing to its left)
            int H = max(Ht[k], F);
            if (c0 + k > g.m) H = SFE_NEG;
            if (TB) {                                     // sign bits shifted in, newest nibble lowest: column k ends at bits 4(3-k)..
                const int Hgl = Hprev - OX;
                nibs = __funnelshift_l((uint32_t)(M[k] - H), nibs, 1);
                nibs = __funnelshift_l((uint32_t)(E[k] - H), nibs, 1);
                nibs = __funnelshift_l((uint32_t)(Hu[k] - E[k]), nibs, 1);
                nibs = __funnelshift_l((uint32_t)(Hgl - F), nibs, 1);
            }
            Hprev = H;
            Hc[k] = H;
            ph[k] = k == 0 ? H : max(ph[k - 1], H);
        }
        // Lambda = 0 (R4, the serial reading): the threshold of (i, j) uses the best over alive cells that precede it in
        // row-major order = max(best of rows < i, prefix maximum of H over the columns left of j): a cell that raises the
        // best is alive by construction and a dead one lies below it, so the maximum may run over every computed H.
        int pb0 = BK_NINF, Bprev = 0;
        if (LAG0) {
            const int incl2 = warp_scan_max(ph[BK_CPT - 1], lane);
            int excl2 = __shfl_up_sync(FULL, incl2, 1);
            if (lane == 0) excl2 = BK_NINF;
            if (lane == 31) sh.tot2[rank] = incl2;
            __syncthreads();                                                                  // B1b
            const int t2 = lane < BK_WARPS ? sh.tot2[lane] : BK_NINF;
            const int carry2 = __reduce_max_sync(FULL, lane < rank ? t2 : BK_NINF);
            pb0 = max(excl2, carry2);
            Bprev = i > 0 ? sh.cum[(i - 1) & 63] : 0;
        }
#pragma unroll
        for (int k = 0; k < BK_CPT; k++) {
            const int H = Hc[k];
            bool alive;
            if (LAG0) {
                const int pb = k == 0 ? pb0 : max(pb0, ph[k - 1]);
                alive = p.ydrop_inf ? H >= SFE_T_INF : H >= max(Bprev, pb) - p.Y;
            } else alive = H >= T;                        // R5
            Hu[k] = alive ? H - OX : SFE_NEG;
            Eu[k] = E[k];
            if (alive) {
                if (H > hmax) { hmax = H; hcol = c0 + k; }
                cl = min(cl, c0 + k); cr = c0 + k;
            }
        }
        // ---- row statistics ----
        const int hm = __reduce_max_sync(FULL, hmax);
        const int hc = __reduce_min_sync(FULL, hmax == hm ? hcol : 0x7fffffff);
        const int wl = __reduce_min_sync(FULL, cl);
        const int wr = __reduce_max_sync(FULL, cr);
        if (lane == 31) sh.edge[warp] = Hu[BK_CPT - 1];
        if (lane == 0) { sh.wmax[warp] = hm; sh.wcol[warp] = hc; sh.wL[warp] = wl; sh.wR[warp] = wr; }
        __syncthreads();                                                                      // B2
        const int L = __reduce_min_sync(FULL, lane < BK_WARPS ? sh.wL[lane] : 0x7fffffff);
        const int R = __reduce_max_sync(FULL, lane < BK_WARPS ? sh.wR[lane] : -1);
        if (R < 0) break;                                 // first row without an alive cell: all later rows are dead
        rows_done = i + 1;
        cells += (unsigned long long)(R - L + 1);
        max_width = max(max_width, R - L + 1);
        // ---- row record: the warps between the first and the last alive column store 16 bits per thread ----
        if (TB && tb_ok) {
            const int r_lo = (L - ws) >> 7, r_hi = (R - ws) >> 7;
            const int nw = 16 * (r_hi - r_lo + 1);
            if (wpos + nw + 2 > BK_CHUNK_WORDS) {         // next chunk (uniform decision)
                if (warp == 0) {
                    if (cur_chunk >= 0 && lane == 0) p.pool[(size_t)cur_chunk * BK_CHUNK_WORDS] = (uint32_t)wpos;
                    const int nc = chunk_pop(p.free_ring, p.ring_state, p.n_chunks, lane);
                    if (lane == 0) { sh.new_chunk = nc; if (nc >= 0) p.chunk_prev[nc] = cur_chunk; if (nc == -2) atomicAdd(&p.counters[CNT_RING_DROPS], 1ULL); }
                }
                __syncthreads();
                const int nc = sh.new_chunk;
                __syncthreads();
                if (nc < 0) tb_ok = false;
                else { cur_chunk = nc; wpos = 1; }
            }
            if (tb_ok) {
                uint32_t *rec = p.pool + (size_t)cur_chunk * BK_CHUNK_WORDS + wpos;
                if (rank >= r_lo && rank <= r_hi) ((uint16_t *)rec)[32 * (rank - r_lo) + lane] = (uint16_t)nibs;
                if (tid == 0) { rec[nw] = (uint32_t)(ws + 128 * r_lo); rec[nw + 1] = (uint32_t)nw; }
                wpos += nw + 2; n_words += nw + 2;
            }
        }
        // ---- warp 0: cumulative best (for T of row i + 32) and the first maximum (R7) ----
        if (warp == 0) {
            const int wm = lane < BK_WARPS ? sh.wmax[lane] : SFE_NEG;
            const int gm = __reduce_max_sync(FULL, wm);
            const int gc = __reduce_min_sync(FULL, (lane < BK_WARPS && wm == gm) ? sh.wcol[lane] : 0x7fffffff);
            if (lane == 0) {
                const int prev = i > 0 ? sh.cum[(i - 1) & 63] : 0;
                sh.cum[i & 63] = max(prev, gm);
                if (gm > sh.best) { sh.best = gm; sh.best_i = i; sh.best_j = gc; sh.best_chunk = cur_chunk; sh.best_wpos = wpos; }
            }
        }
        // ---- next row's window ----
        if (R - (L & ~127) >= BK_WIN - 1) { wide = true; break; }  // an alive cell in the last column the next window could hold
        ws_prev = ws;
        ws = L & ~127;
    }
    __syncthreads();
    if (TB && cur_chunk >= 0 && tid == 0) p.pool[(size_t)cur_chunk * BK_CHUNK_WORDS] = (uint32_t)wpos;

    out.score = sh.best; out.end_i = sh.best_i; out.end_j = sh.best_j; out.cells = cells;
    out.status = (wide ? (LAG0 ? SFE_ST_BAND_LIMIT : SFE_ST_WIDE_PENDING) : 0u) | ((TB && !tb_ok) ? SFE_ST_PASS_OVERFLOW : 0u) | SFE_ST_BLOCK |
                 (limit ? SFE_ST_SCORE_LIMIT : 0u);
    out.n_strips = rows_done; out.n_rec = (int)(n_words >> 6); out.steps = rows_done; out.max_steps = max_width;
    // ---- a8: warp 0 walks the row log and stages the ops; then the chunks go back to the ring ----
    if (warp == 0) {
        if (TB && tb_ok && !wide && !limit) {
            bool ops_ok = true;
            if (!block_walk(p, sh, sh.best_i, sh.best_j, sh.best_chunk, sh.best_wpos, lane, out.ops_seg, out.n_ops, ops_ok))
                out.status |= SFE_ST_INTERNAL;
            if (!ops_ok) out.status |= SFE_ST_OPS_OVERFLOW;
        }
        if (TB) {
            __threadfence();
            __syncwarp();
            int cc = cur_chunk;
            while (cc >= 0) { const int prev = __ldcg(p.chunk_prev + cc); chunk_push(p.free_ring, p.ring_state, p.n_chunks, cc, &p.counters[CNT_RING_DROPS], lane); cc = prev; }
        }
        unsigned smid, wslot;
        asm("mov.u32 %0, %%smid;" : "=r"(smid));
        asm("mov.u32 %0, %%warpid;" : "=r"(wslot));
        out.cycles = clock64() - clk0; out.smid = smid; out.wslot = wslot;
        if (lane == 0) {
            p.halves[hid] = out;
            atomicAdd(&p.counters[CNT_STEPS], (unsigned long long)rows_done);
            if (TB) atomicAdd(&p.counters[CNT_TBBYTES], (unsigned long long)n_words * 4ULL);
            if (TB && !tb_ok) atomicAdd(&p.counters[CNT_OVERFLOW], 1ULL);
            if (wide && !LAG0) atomicAdd(&p.counters[CNT_WIDE], 1ULL);
            atomicAdd(&p.counters[CNT_BLOCK_HALVES], 1ULL);
        }
    }
}

// Persistent CTAs: each pulls the next half from the ticket list (longest bin first).
template <bool TB, bool LAG0>
__global__ void __launch_bounds__(BK_THREADS, 2) ydrop_block_kernel(const YdParams p)
{
    __shared__ BkShared sh;
    __shared__ unsigned long long tk_s;
    for (;;) {
        if (threadIdx.x == 0) tk_s = atomicAdd(&p.counters[CNT_TICKET], 1ULL);
        __syncthreads();
        const long long tk = (long long)tk_s;
        __syncthreads();
        if (tk >= p.n_tickets) break;
        block_half<TB, LAG0>(p, p.tickets[tk], sh);
        __syncthreads();
    }
}

int sfe_launch_ydrop_block(const YdParams &p, bool want_tb, int n_sm, cudaStream_t st)
{
    long long blocks = p.n_tickets < 2LL * n_sm ? p.n_tickets : 2LL * n_sm;      // two CTAs of 8 warps per SM
    if (blocks < 1) blocks = 1;
    if (p.lag0) {
        if (want_tb) SFE_KL ydrop_block_kernel<true, true><<<(unsigned)blocks, BK_THREADS, 0, st>>>(p);
        else SFE_KL ydrop_block_kernel<false, true><<<(unsigned)blocks, BK_THREADS, 0, st>>>(p);
    } else {
        if (want_tb) SFE_KL ydrop_block_kernel<true, false><<<(unsigned)blocks, BK_THREADS, 0, st>>>(p);
        else SFE_KL ydrop_block_kernel<false, false><<<(unsigned)blocks, BK_THREADS, 0, st>>>(p);
    }
    SFE_LAUNCH_CHECK();
}
