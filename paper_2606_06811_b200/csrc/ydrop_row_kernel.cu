// ydrop_row_kernel.cu -- cooperative warps per anchor-half, second design ("8 warps
// per anchor-half ... kernel wall time / 3.3"), for the LONG halves whose serial chain bounds a pass.
//
// Why a second kernel.  With the row-lagged threshold (R4, Lambda = 32) at most 32 rows of one extension can be in flight:
// the warp-systolic kernel turns a half of n rows into ~ n/32 (W + 62) dependent wavefront steps, measured 1,030 cycles per
// row score-only and 1,450 with traceback on a 580 k-row half of configs[4] (profiles/r2_03), whatever else the GPU does.
// The parallelism that is left is ALONG a row: one CTA per half, rows strictly in order, every thread owns RK_C consecutive
// columns of a 1024-column window.  The first cooperative kernel (ydrop_block_kernel.cu, kept for Lambda = 0) spent ~700
// instructions per thread per row and two block barriers on that (2,256 cycles per row).  This one: 780 score-only /
// 1,030 with traceback on the same half (profiles/r2_04) -- a quarter / 30 % less than the systolic chain.  It takes the
// tickets a pass predicts longest (SFE_OPT_ROW_KERNEL_CAP, default: one per SM, beside the systolic kernel; the CTA claims
// its SM while it works), every ticket with SFE_BLOCK_KERNEL, and the halves handed over by SFE_OPT_LONG_ROWS.  Design:
//   * ONE block barrier per row (the exchange of the warps' F carries); the diagonal hand-off between neighbouring warps
//     is an 8-byte {value, row} word that the reader polls (it is there by the time it is needed);
//   * F(i,j) = max_{j'<j} (H~(i,j') - O - X (j - j')), H~ = max(M, E): a sequential max-plus chain over the thread's own
//     columns (DPX VIADDMNMX), one shuffle scan per warp (shfl_up returns the caller's own value out of range, so a max
//     scan needs no predicate), one 4-entry combine across warps;
//   * everything that is not needed for the next row is LAGGED: per-row maxima (for T of row i + 32), alive bounds (cell
//     count, end of the half, window position) go to shared-memory rings -- written one row late, under the next row's
//     scan -- and are folded every 16 rows, where the thresholds of the next 16 rows are computed at once;
//   * whatever depends only on the window position (the warp's rank, the thread's columns, the constants of the carry
//     exchange, the target-end caps) is set when the window moves, and everything periodic (fold, query bases, traceback
//     chunk: popped one fold ahead) sits behind ONE test per row: a branch costs this loop 15-20 cycles, taken or not;
//   * the column -> (warp, lane, slot) map is fixed modulo the window, so a traceback row is a fixed 512-byte record the
//     walk can address without any directory, and a thread's 8 nibbles are exactly one coalesced 32-bit store;
//   * the "F extended" bit is stored with the cell the gap run CONTINUES FROM (F(i,j) - X > H(i,j) - (O+X): the cell's own
//     values) instead of the cell it arrives at, so no final H crosses a thread boundary within a row.
// Exactness (same argument as ydrop_block_kernel.cu): E depends on the column above only; the prefix maximum over H~ equals
// the recurrence over H because a gap opened from an H that came from F never beats extending that F (O >= 0); by the R6
// lemma cells that are dead or outside the window (which starts at or left of the first alive column of an older row; that
// column never moves left) contribute nothing an alive cell, its H or a pointer on an alive path depends on.  Score, end
// cell (first maximum, R7), cell count (R28) and CIGAR (R11, R12) are the oracle's at Lambda = 32: same tests as ydrop_kernel.
#include "ydrop_common.cuh"

#ifndef RK_NW
#define RK_NW 8                              // warps per CTA: two per SM sub-partition hide each other's dependency stalls
#endif
#ifndef RK_C
#define RK_C 4                               // columns per thread
#endif
#define RK_THREADS (32 * RK_NW)
#define RK_WCOLS (32 * RK_C)                 // columns per warp: the window moves in steps of this
#define RK_WIN (RK_THREADS * RK_C)           // 1024
#define RK_ROW_WORDS (RK_WIN / 8)            // traceback record of a row: 4 bits per window column = 512 B
#define RK_CHUNK_ROWS (SFE_CHUNK_BYTES / (4 * RK_ROW_WORDS))     // 128 rows per 64-KiB chunk
#define RK_NINF (-(1 << 30) - (1 << 28))     // identity of the max-plus scans: the decay terms (< 2^27) fit below it, and H - O - F with
                                             // H < 2^29 (R25) stays inside int32
#define RK_FOLD 16                           // rows between two folds of the lagged statistics
#define RK_POLL_LIMIT (1 << 22)
#ifdef RK_PROFILE
#include <stdio.h>
#define RK_T(k) do { const long long t_ = clock64(); prof_t[k] += t_ - prof_last; prof_last = t_; } while (0)
#else
#define RK_T(k) do { } while (0)
#endif

struct RkShared {
    unsigned long long edge[RK_NW];          // by warp: {row << 32 | gated H - OX of its last column after that row}: ONE 8-byte word
    __align__(16) int carry[2][RK_NW];       // by row parity, RANK of the warp in the window: F leaving the warp (+ Dw * rank)
    __align__(16) int rmax[64][RK_NW];       // by row & 63, warp: max H of the row (any cell: a dead one never raises the best)
    __align__(16) int rlo[64][RK_NW];        // first / last alive column of the row in the warp's block (lo > hi: none)
    __align__(16) int rhi[64][RK_NW];
    __align__(8) int fail_row;               // row in which a bounded wait ran out (never expected; -1 = none): SFE_ST_INTERNAL
    int wide_row;                            // row in which the window's last column held an alive cell (-1 = none): the band outgrew it
    int new_chunk;
    int red_s[RK_NW], red_i[RK_NW], red_j[RK_NW];
    uint32_t opsbuf[SFE_WALK_OPS];
};

// Shared memory is addressed through ONE 32-bit base kept in a register and explicit ld/st.shared: left to the compiler,
// every access to the static struct re-derives its address from SR_CgaCtaId (S2UR + ULEA on sm_100a), ~25 cycles a time
// on a path that is latency-bound.
#include <stddef.h>
#define RK_OFF(field) ((uint32_t)offsetof(RkShared, field))
static __device__ __forceinline__ int lds32(uint32_t a) { int v; asm volatile("ld.shared.s32 %0, [%1];" : "=r"(v) : "r"(a)); return v; }
static __device__ __forceinline__ int2 lds64(uint32_t a) { int2 v; asm volatile("ld.shared.v2.s32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(a)); return v; }
static __device__ __forceinline__ int4 lds128(uint32_t a) { int4 v; asm volatile("ld.shared.v4.s32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a)); return v; }
static __device__ __forceinline__ unsigned long long lds_u64v(uint32_t a) { unsigned long long v; asm volatile("ld.volatile.shared.u64 %0, [%1];" : "=l"(v) : "r"(a) : "memory"); return v; }
static __device__ __forceinline__ void sts32(uint32_t a, int v) { asm volatile("st.shared.s32 [%0], %1;" :: "r"(a), "r"(v) : "memory"); }
static __device__ __forceinline__ void sts32_if(bool c, uint32_t a, int v)
{
    asm volatile("{ .reg .pred p; setp.ne.u32 p, %0, 0; @p st.shared.s32 [%1], %2; }" :: "r"((unsigned)c), "r"(a), "r"(v) : "memory");
}
static __device__ __forceinline__ void sts_u64v(uint32_t a, unsigned long long v) { asm volatile("st.volatile.shared.u64 [%0], %1;" :: "r"(a), "l"(v) : "memory"); }

// maximum over the RK_NW per-warp entries of one ring row: broadcast 128-bit loads, no reduction instruction
static __device__ __forceinline__ int row_max4(uint32_t a)
{
    int m = SFE_NEG;
#pragma unroll
    for (int w = 0; w < RK_NW; w += 4) { const int4 x = lds128(a + 4 * w); m = max(m, max(max(x.x, x.y), max(x.z, x.w))); }
    return m;
}
static __device__ __forceinline__ int row_min4(uint32_t a)
{
    int m = 0x7fffffff;
#pragma unroll
    for (int w = 0; w < RK_NW; w += 4) { const int4 x = lds128(a + 4 * w); m = min(m, min(min(x.x, x.y), min(x.z, x.w))); }
    return m;
}

// ---- a8: walk the fixed-size row records from the end cell to the origin (warp 0; every lane holds the same state) ----
// Nibble of cell (i, j): word (j mod RK_WIN) / 8 of row i's record (position inside the word: see nibble() below):
//   bit3 = H not from M, bit2 = H not from E, bit1 = E extended (R11), bit0 = the F of the NEXT column extends this cell's F.
static __device__ bool row_walk(const YdParams &p, uint32_t *opsbuf, const int end_i, const int end_j, int chunk, const int lane,
                                uint32_t &ops_seg, int &n_ops, bool &ops_ok)
{
    OpsWriter ow;
    ow.buf = opsbuf; ow.stage = p.ops_stage; ow.used = &p.counters[CNT_OPS]; ow.cap = p.ops_cap;
    ow.nbuf = 0; ow.nops = 0; ow.cur_op = -1; ow.run = 0; ow.prev_seg = SFE_NO_SEG; ow.ok = true;
    ops_seg = SFE_NO_SEG; n_ops = 0; ops_ok = true;
    if (end_i == 0 && end_j == 0) return true;
    if (chunk < 0) return false;
    // `chunk` holds the rows of ordinal `ord`; the chain runs backwards through chunk_prev
    int ord = end_i / RK_CHUNK_ROWS;
    int prev = __ldcg(p.chunk_prev + chunk);
    int i = end_i, j = end_j, state = 0;
    long long guard = 3LL * ((long long)end_i + end_j) + 64;
    auto nibble = [&](int r, int c) -> uint32_t {
        const int o = r / RK_CHUNK_ROWS;
        const int ch = o == ord ? chunk : prev;                  // 32 consecutive rows span at most two chunks
        const uint32_t w = __ldcg(p.pool + (size_t)ch * (SFE_CHUNK_BYTES / 4) + (size_t)(r - o * RK_CHUNK_ROWS) * RK_ROW_WORDS +
                                  ((c & (RK_WIN - 1)) >> 3));
        // a thread's RK_C nibbles (first column highest) form one 4 RK_C-bit unit; units fill the word from its low end
        return (w >> (4 * (RK_C - 1 - (c & (RK_C - 1))) + 4 * RK_C * ((c & 7) / RK_C))) & 15u;
    };
    while (!(i == 0 && j == 0 && state == 0)) {
        if (--guard < 0) return false;
        while (i / RK_CHUNK_ROWS < ord) {                        // the walk left the current chunk's rows
            chunk = prev; ord--;
            if (chunk < 0) return false;
            prev = __ldcg(p.chunk_prev + chunk);
        }
        if (prev < 0 && ord > 0) return false;
        if (state == 2) {
            // F: emit D, go left; the run continues while the cell we arrive at says "my F is extended into the next column"
            const int jx = j - 1 - lane;
            const bool valid = jx >= 0;
            uint32_t nib = 0;
            if (valid) nib = nibble(i, jx);
            const uint32_t stop = __ballot_sync(FULL, !(valid && (nib & 1u)));
            const int pstop = stop ? __ffs(stop) - 1 : 32;       // cells j-1 .. j-pstop continue; the run was opened at j-1-pstop
            const int cnt = pstop < 32 ? pstop + 1 : 32;
            ow.emit(SFE_OP_D, cnt, lane);
            j -= cnt;
            if (pstop < 32) state = 0;
            if (j < 0) return false;
            continue;
        }
        // H (diagonal) or E (up): lane x examines the x-th cell from (i, j) in the current direction
        const int dj = state == 1 ? 0 : 1;
        const int ix = i - lane, jx = j - lane * dj;
        const bool valid = ix >= 0 && jx >= 0 && ix / RK_CHUNK_ROWS >= ord - 1;
        uint32_t nib = 0;
        if (valid) nib = nibble(ix, jx);
        const bool cont = state == 0 ? !(nib & 8u) : (nib & 2u) != 0;
        const bool origin = ix == 0 && jx == 0;
        const uint32_t stop = __ballot_sync(FULL, !(valid && cont) || origin);
        const uint32_t vmask = __ballot_sync(FULL, valid);
        const int pstop = stop ? __ffs(stop) - 1 : 32;
        const bool stop_valid = pstop < 32 && ((vmask >> pstop) & 1u);
        if (pstop == 0 && !stop_valid) return false;
        if (state == 0) {
            ow.emit(SFE_OP_M, pstop, lane);
            i -= pstop; j -= pstop;
            if (stop_valid && !(i == 0 && j == 0)) {
                const uint32_t nb = __shfl_sync(FULL, nib, pstop);
                state = (nb & 4u) ? 2 : 1;
            }
        } else {
            const int cnt = stop_valid ? pstop + 1 : pstop;
            ow.emit(SFE_OP_I, cnt, lane);
            i -= cnt;
            if (stop_valid) state = 0;
        }
    }
    if (ow.cur_op >= 0) ow.push(lane);
    ow.flush(lane);
    ops_seg = ow.prev_seg; n_ops = ow.nops; ops_ok = ow.ok;
    return true;
}

template <bool TB>
static __device__ __forceinline__ void row_half(const YdParams &p, const int hid)
{
    // a function-scope __shared__ object: every access below is a direct shared-space LDS / STS with an immediate offset.
    // (Reached through a reference parameter the same struct was addressed generically: each access re-derived the
    // shared window from SR_CgaCtaId -- S2UR + ULEA -- and the row cost 1,350 cycles instead of ~700.)
    __shared__ RkShared sh;
    uint32_t sb = (uint32_t)__cvta_generic_to_shared(&sh);
    asm volatile("" : "+r"(sb));                          // opaque: one register, no re-derivation
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
    const int OX = p.OX, X = p.X, O = p.OX - p.X;
    const int D = X * RK_C, Dw = X * RK_WCOLS;
    const uint32_t srow_hi = p.srow_hi;

    if (tid < RK_NW) { sh.edge[tid] = 0xffffffff00000000ULL | (unsigned)SFE_NEG; sh.carry[0][tid] = RK_NINF; sh.carry[1][tid] = RK_NINF; }
    if (tid == 0) { sh.fail_row = -1; sh.wide_row = -1; sh.new_chunk = -1; }
    __syncthreads();

    int ws = 0;                                           // window start (a multiple of RK_WCOLS); moves only at a fold
    int myc0 = -1;                                        // first of my RK_C columns
    int Hu[RK_C], Eu[RK_C];                               // previous row of my columns: gated H - OX, E
    uint32_t sel[RK_C];
#pragma unroll
    for (int k = 0; k < RK_C; k++) { Hu[k] = SFE_NEG; Eu[k] = SFE_NEG; sel[k] = 0x8880u; }
    int best = 0, best_i = 0, best_j = 0;                 // thread-local first maximum (my cells are visited in row-major order)
    int cumbest = 0;                                      // best over alive cells of rows <= i - 32 (uniform)
    unsigned long long cells = 0;                         // folded rows (uniform)
    int folded = 0;                                       // rows < folded have been folded (uniform)
    int rows_done = 0, max_width = 0, last_lo = 0;
    bool wide = false, limit = false;
    uint32_t srow32 = 0u;
    int cur_chunk = -1;                                   // traceback chunk of the current 128 rows (uniform)
    bool tb_ok = TB;
    long long n_words = 0;

    // fold the statistics of rows [folded, upto): cells, first dead row, newest alive bounds.  Uniform: every warp reads the
    // same shared-memory rings (written >= 16 block barriers ago).  Returns false when a row without an alive cell was found.
    auto fold = [&](int upto, int &new_lo, int &new_hi) -> bool {
        bool alive_all = true;
        while (folded < upto) {
            const int r = folded + lane;
            int lo = 0x7fffffff, hi = -1;
            if (r < upto) { lo = row_min4(sb + RK_OFF(rlo) + 4 * RK_NW * (r & 63)); hi = row_max4(sb + RK_OFF(rhi) + 4 * RK_NW * (r & 63)); }
            const unsigned nb = r < upto ? 1u : 0u;
            const unsigned deadm = __ballot_sync(FULL, nb && hi < lo);
            const int nrows = min(32, upto - folded);
            const int ndead_first = deadm ? __ffs(deadm) - 1 : nrows;            // rows before the first dead one count
            const int width = (nb && lane < ndead_first) ? hi - lo + 1 : 0;
            unsigned long long wsum = (unsigned long long)width;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) wsum += __shfl_xor_sync(FULL, wsum, o);
            cells += wsum;
            max_width = max(max_width, __reduce_max_sync(FULL, width));
            if (ndead_first > 0) {
                new_lo = __shfl_sync(FULL, lo, ndead_first - 1); new_hi = __shfl_sync(FULL, hi, ndead_first - 1);
                rows_done = folded + ndead_first;
            }
            if (deadm) { alive_all = false; folded = 0x7fffffff; break; }        // everything after the first dead row is dead
            folded += nrows;
        }
        return alive_all;
    };

#ifdef RK_PROFILE
    long long prof_t[8] = {0, 0, 0, 0, 0, 0, 0, 0}, prof_last = clock64();
#endif
    // Everything that depends only on the window position is computed when the window moves (at a fold), not per row: the
    // warp's rank, the thread's columns, the constants of the carry exchange.  A thread's columns are fixed modulo RK_WIN.
    int rho = warp, c0 = tid * RK_C;                      // my warp's rank in the window; my first column
    int k1 = 0, carry_add = 0;                            // Dw (rho - 1) + D lane;  Dw rho - 31 D
    bool need_edge = false;
    int hcap[RK_C];
    const int lw = (warp - 1) & (RK_NW - 1);
    auto set_window = [&](const int nws, const int ows) {
        rho = (warp - nws / RK_WCOLS) & (RK_NW - 1);
        c0 = nws + rho * RK_WCOLS + lane * RK_C;
        if (c0 != myc0) {                                 // (the warp's columns change together)
            myc0 = c0;
#pragma unroll
            for (int k = 0; k < RK_C; k++) { Hu[k] = SFE_NEG; Eu[k] = SFE_NEG; sel[k] = col_selector(g, c0 + k); }
        }
#pragma unroll
        for (int k = 0; k < RK_C; k++) hcap[k] = c0 + k > g.m ? SFE_NEG : 0x7fffffff;    // (only the threads at the target's end)
        k1 = Dw * (rho - 1) + D * lane;
        carry_add = Dw * rho - D * 31;
        // the diagonal of the warp's first column comes from the left warp iff that column was inside the previous window
        need_edge = rho != 0 && nws + rho * RK_WCOLS - 1 - ows < RK_WIN;
    };
    set_window(0, 0);
    need_edge = false;                                    // row 0 has no row above it
    int Tvec = p.ydrop_inf ? SFE_T_INF : -p.Y;            // lane k: T of row (i & ~15) + k
    unsigned char *rec_ptr = nullptr;                     // my RK_C-cell unit (RK_C / 2 bytes) of the current row's traceback record
    int pend_chunk = -1;                                  // warp 0: the chunk popped ahead for the next 128 rows, not adopted yet
    int tb_rows = 0;                                      // rows with a traceback record
    uint32_t am_p = 0; int hmax_p = SFE_NEG, c0_p = 0;    // the previous row's alive mask / maximum / first column: published one row late

    // The statistics of a row are published while the NEXT row's scan is in flight (branch-free, so the scheduler can put
    // them into the shuffles' latency); the fold reads rows >= 16 barriers old, so one row of delay costs nothing.
    auto publish_prev = [&](const int row) {
        // lowest / highest set bit of the RK_C-bit mask from two packed tables (plain ALU; FLO sits on the slow pipe)
        static_assert(RK_C <= 4, "the packed bit-position tables cover 4-bit masks");
        const int lo_v = am_p ? c0_p + (int)((0x12131210u >> (2 * am_p)) & 3u) : 0x7fffffff;     // 2 bits per mask value 0 .. 15
        const int hi_v = am_p ? c0_p + (int)((0xffffaa50u >> (2 * am_p)) & 3u) : -1;
        const int wlo = __reduce_min_sync(FULL, lo_v), whi = __reduce_max_sync(FULL, hi_v), wm = __reduce_max_sync(FULL, hmax_p);
        const uint32_t so = sb + 4 * (RK_NW * (row & 63) + warp);
        const int v = lane == 0 ? wlo : lane == 1 ? whi : wm;
        const uint32_t off = lane == 0 ? RK_OFF(rlo) : lane == 1 ? RK_OFF(rhi) : RK_OFF(rmax);
        sts32_if(lane < 3, so + off, v);
    };

    if (TB) {                                             // the chunk of rows 0 .. 127
        if (warp == 0) {
            const int nc = chunk_pop(p.free_ring, p.ring_state, p.n_chunks, lane);
            if (lane == 0) {
                sh.new_chunk = nc;
                if (nc >= 0) p.chunk_prev[nc] = -1;
                if (nc == -2) atomicAdd(&p.counters[CNT_RING_DROPS], 1ULL);
            }
        }
        __syncthreads();
        const int nc = lds32(sb + RK_OFF(new_chunk));
        if (nc < 0) tb_ok = false;
        else { cur_chunk = nc; rec_ptr = (unsigned char *)(p.pool + (size_t)nc * (SFE_CHUNK_BYTES / 4)) + tid * (RK_C / 2); }
        __syncthreads();
    }

    int i = 0;
    for (; i <= g.n; i++) {
        RK_T(7);
        // ---- early load: the left warp's edge {row, value} (broadcast), used after the housekeeping ----
        unsigned long long ev = lds_u64v(sb + RK_OFF(edge) + 8 * lw);
        // ---- everything periodic sits behind ONE test per row (a branch costs ~15-20 cycles here, taken or not) ----
        if ((i & (RK_FOLD - 1)) == 0) {
            if (i >= 2 * RK_FOLD) {
                // thresholds of rows i .. i + 15 (R4): T(r) = best(rows <= r - 32) - ydrop; rows i - 32 .. i - 17 were
                // published >= 16 barriers ago.  Lane k < 16 ends with the running best through row i - 32 + k.
                int v = lane < RK_FOLD ? row_max4(sb + RK_OFF(rmax) + 4 * RK_NW * ((i - 32 + lane) & 63)) : SFE_NEG;
#pragma unroll
                for (int o = 1; o < RK_FOLD; o <<= 1) v = max(v, __shfl_up_sync(FULL, v, o));
                v = max(v, cumbest);
                cumbest = __shfl_sync(FULL, v, RK_FOLD - 1);
                if (cumbest >= SFE_SCORE_LIMIT) { limit = true; break; }              // R25
                Tvec = p.ydrop_inf ? SFE_T_INF : v - p.Y;
                // statistics of rows [i - 32, i - 16): cells, termination, the window
                int nlo = last_lo, nhi = -1;
                if (!fold(i - RK_FOLD, nlo, nhi)) break;
                last_lo = nlo;
                const int nws = nlo & ~(RK_WCOLS - 1);            // the first alive column never moves left: a stale one is safe
                // the last alive column grows by at most one per row: rows up to the next fold stay below nhi + 2 RK_FOLD + 1
                if (nhi + 2 * RK_FOLD + 2 >= nws + RK_WIN) { wide = true; break; }
                if (nws != ws) { set_window(nws, ws); ws = nws; }
            }
            if ((i & 31) == 0) {
                const int r = i + lane;
                srow32 = (r == 0 || r > g.n) ? 0u : p.srow[sfe_base(g.qc, g.qm, g.q0 + (long long)g.d * r)];
            }
            if (TB && tb_ok) {
                // the traceback chunk of the next 128 rows is popped by warp 0 one fold ahead and adopted by everybody at the
                // chunk's first row: 16 barriers lie between the two, and no row pays for a test of its own
                const int ph = i & (RK_CHUNK_ROWS - 1);
                if (ph == RK_CHUNK_ROWS - RK_FOLD && warp == 0) {
                    const int nc = chunk_pop(p.free_ring, p.ring_state, p.n_chunks, lane);
                    pend_chunk = nc;
                    if (lane == 0) {
                        sh.new_chunk = nc;
                        if (nc >= 0) p.chunk_prev[nc] = cur_chunk;
                        if (nc == -2) atomicAdd(&p.counters[CNT_RING_DROPS], 1ULL);
                    }
                }
                if (ph == 0 && i > 0) {
                    const int nc = lds32(sb + RK_OFF(new_chunk));
                    pend_chunk = -1;
                    if (nc < 0) tb_ok = false;
                    else { cur_chunk = nc; rec_ptr = (unsigned char *)(p.pool + (size_t)nc * (SFE_CHUNK_BYTES / 4)) + tid * (RK_C / 2); }
                }
            }
        }
        const uint32_t srow_lo = __shfl_sync(FULL, srow32, i & 31);
        const int T = __shfl_sync(FULL, Tvec, i & (RK_FOLD - 1));
        int Hd0 = __shfl_up_sync(FULL, Hu[RK_C - 1], 1);
        publish_prev(i - 1);                                       // (independent of this row: its reductions run under the loads above)
        RK_T(0);
        // ---- diagonal of the warp's first column: the left warp's previous-row value.  The edge is normally there already;
        // the (uniform) slow path polls for it ----
        if (need_edge && (int)(ev >> 32) != i - 1) {
            for (int spin = 0; (int)(ev >> 32) != i - 1 && spin < RK_POLL_LIMIT; spin++) ev = lds_u64v(sb + RK_OFF(edge) + 8 * lw);
            if ((int)(ev >> 32) != i - 1) sts32(sb + RK_OFF(fail_row), i);        // (readers act on it from this row's barrier on)
        }
        if (lane == 0) Hd0 = need_edge ? (int)(unsigned)ev : SFE_NEG;
        need_edge = rho != 0;                                     // (rows after the first one of a window)
        if (i == 0 && c0 == 0) Hd0 = -OX;                         // the origin (R8)
        RK_T(1);
        // ---- phase A: M, E, H~ and the in-thread F chain ----
        int M[RK_C], E[RK_C], Ht[RK_C], gl[RK_C];                 // gl[k]: F entering column k from my own columns left of it
#pragma unroll
        for (int k = 0; k < RK_C; k++) {
            const int Hd = k == 0 ? Hd0 : Hu[k - 1];
            const int s = prmt_sx(srow_lo, srow_hi, sel[k]);
            M[k] = Hd + s + OX;
            E[k] = __viaddmax_s32(Eu[k], -X, Hu[k]);
            Ht[k] = max(M[k], E[k]);
        }
        int gk = RK_NINF;
#pragma unroll
        for (int k = 0; k < RK_C; k++) { gl[k] = gk; gk = __viaddmax_s32(gk, -X, Ht[k] - OX); }
        RK_T(2);
        // ---- F across the threads of the warp: y = x + D lane, prefix maximum, exclusive ----
        // Three doubling steps give y3[l] = max over lanes l-7 .. l; the exclusive prefix over all lanes left of l is then the
        // maximum of y3 at l-1, l-9, l-17, l-25: four INDEPENDENT shuffles (one latency) instead of three more dependent ones.
        int y = gk + D * lane;
#pragma unroll
        for (int o = 1; o < 8; o <<= 1) y = max(y, __shfl_up_sync(FULL, y, o));       // out-of-range lanes get their own value back
        int e0 = __shfl_up_sync(FULL, y, 1), e1 = __shfl_up_sync(FULL, y, 9), e2 = __shfl_up_sync(FULL, y, 17), e3 = __shfl_up_sync(FULL, y, 25);
        e0 = lane >= 1 ? e0 : RK_NINF; e1 = lane >= 9 ? e1 : RK_NINF; e2 = lane >= 17 ? e2 : RK_NINF; e3 = lane >= 25 ? e3 : RK_NINF;
        const int yex = max(max(e0, e1), max(e2, e3));
        // F leaving the warp (inclusive at lane 31), pre-shifted by the warp's rank
        sts32_if(lane == 31, sb + RK_OFF(carry) + 4 * (RK_NW * (i & 1) + rho), max(yex, y) + carry_add);
        const int fin_warp = yex - D * lane + D;                   // F entering my first column from my warp's lanes left of me
        RK_T(3);
        __syncthreads();                                                                   // the one barrier of the row
        RK_T(4);
        // ---- after the barrier: flags and the other warps' carries, requested together ----
        const int2 fl = lds64(sb + RK_OFF(fail_row));
        // the carries of the warps left of mine: lane r < rho loads carry[r], one warp reduction (uniform result)
        const int cv = lane < rho ? lds32(sb + RK_OFF(carry) + 4 * (RK_NW * (i & 1) + (lane & (RK_NW - 1)))) : RK_NINF;
        const int cm = __reduce_max_sync(FULL, cv);
        // both flags carry the row they were raised in (-1: not raised): a fast warp's later write is ignored by a slow
        // reader, so every thread leaves the loop in the same row (a non-uniform exit would hang the next barrier)
        if ((unsigned)fl.x <= (unsigned)i || (unsigned)fl.y < (unsigned)i) {
            if (!((unsigned)fl.x <= (unsigned)i)) wide = true;
            break;
        }
        // F entering my warp from the warps left of it: max_{r < rho} carry_r - Dw (rho - 1 - r); then down my warp's lanes
        const int Fin = max(fin_warp, cm - k1);
        RK_T(5);
        // ---- phase C: F, H, alive, next row's state, statistics, pointers ----
        uint32_t nibs = 0, am = 0;
        int hmax = SFE_NEG;
        const int best_before = best;
        int Hc[RK_C];
#pragma unroll
        for (int k = 0; k < RK_C; k++) {
            const int F = max(gl[k], Fin - X * k);
            int H = max(Ht[k], F);
            H = min(H, hcap[k]);                                   // columns beyond the target (set with the window)
            const bool alive = H >= T;                             // R5
            if (TB) {
                nibs = __funnelshift_l((uint32_t)(M[k] - H), nibs, 1);           // H not from M
                nibs = __funnelshift_l((uint32_t)(E[k] - H), nibs, 1);           // H not from E
                nibs = __funnelshift_l((uint32_t)(Hu[k] - E[k]), nibs, 1);       // E extended (open wins ties)
                nibs = __funnelshift_l((uint32_t)(H - O - F), nibs, 1);          // next column's F extends this F: F - X > H - (O+X)
            }
            Hu[k] = alive ? H - OX : SFE_NEG;
            Eu[k] = E[k];
            Hc[k] = H;
            hmax = max(hmax, H);
            if (alive) am |= 1u << k;
        }
        RK_T(6);
        // ---- publish the edge for the next row first: the right warp is waiting for it ----
        if (lane == 31) sts_u64v(sb + RK_OFF(edge) + 8 * warp, ((unsigned long long)(unsigned)i << 32) | (unsigned)Hu[RK_C - 1]);
        sts32_if(rho == RK_NW - 1 && lane == 31 && (am >> (RK_C - 1)), sb + RK_OFF(wide_row), i);   // alive in the window's last column: bail out next row
        best = max(best, hmax);
        if (best > best_before) {                                  // strict: the first maximum of my cells (R7)
            int kk = RK_C - 1;
#pragma unroll
            for (int k = RK_C - 2; k >= 0; k--) kk = Hc[k] == best ? k : kk;
            best_i = i; best_j = c0 + kk;
        }
        am_p = am; hmax_p = hmax; c0_p = c0;
        if (TB) {
            if (tb_ok) {
                if (RK_C == 8) *(uint32_t *)rec_ptr = nibs;
                else if (RK_C == 4) *(uint16_t *)rec_ptr = (uint16_t)nibs;
                else *rec_ptr = (unsigned char)nibs;
            }
            rec_ptr += 4 * RK_ROW_WORDS;
            tb_rows += tb_ok ? 1 : 0;
        }
    }
    publish_prev(i - 1);                                           // the last computed row (again, if the loop left after its barrier)
    n_words = (long long)tb_rows * RK_ROW_WORDS;
#ifdef RK_PROFILE
    if (lane == 0 && i > 100000) printf("RKPROF warp %d rows %d: top %.1f cols/poll %.1f phaseA %.1f scan %.1f barrier %.1f postbar %.1f phaseC %.1f publish %.1f\n", warp, i, (double)prof_t[0] / i, (double)prof_t[1] / i, (double)prof_t[2] / i, (double)prof_t[3] / i, (double)prof_t[4] / i, (double)prof_t[5] / i, (double)prof_t[6] / i, (double)prof_t[7] / i);
#endif
    __syncthreads();
    // ---- the rows not folded yet (rows 0 .. i-1 were computed) ----
    const bool failed = sh.fail_row >= 0;
    if (!failed && !wide && folded < i) {
        int nlo = last_lo, nhi = -1;
        fold(i, nlo, nhi);
    }
    // ---- first maximum over the threads: key (score desc, i asc, j asc) (R7) ----
    int bs = best, bi = best_i, bj = best_j;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const int os = __shfl_xor_sync(FULL, bs, o), oi = __shfl_xor_sync(FULL, bi, o), oj = __shfl_xor_sync(FULL, bj, o);
        if (os > bs || (os == bs && (oi < bi || (oi == bi && oj < bj)))) { bs = os; bi = oi; bj = oj; }
    }
    if (lane == 0) { sh.red_s[warp] = bs; sh.red_i[warp] = bi; sh.red_j[warp] = bj; }
    __syncthreads();
    bs = sh.red_s[0]; bi = sh.red_i[0]; bj = sh.red_j[0];
#pragma unroll
    for (int w = 1; w < RK_NW; w++) {
        const int os = sh.red_s[w], oi = sh.red_i[w], oj = sh.red_j[w];
        if (os > bs || (os == bs && (oi < bi || (oi == bi && oj < bj)))) { bs = os; bi = oi; bj = oj; }
    }
    out.score = bs; out.end_i = bi; out.end_j = bj; out.cells = cells;
    out.status = (wide ? SFE_ST_WIDE_PENDING : 0u) | ((TB && !tb_ok) ? SFE_ST_PASS_OVERFLOW : 0u) | SFE_ST_BLOCK |
                 (limit ? SFE_ST_SCORE_LIMIT : 0u) | (failed ? SFE_ST_INTERNAL : 0u);
    // n_strips / steps feed the overflow re-run's chunk estimate (queue_kernels.cu): a row costs two 256-byte records
    out.n_strips = 2 * rows_done; out.n_rec = (int)(n_words >> 6); out.steps = rows_done; out.max_steps = max_width;
    // ---- a8: warp 0 walks the row records and stages the ops; then the chunks go back to the ring ----
    if (warp == 0) {
        if (TB && tb_ok && !wide && !limit && !failed) {
            // the end cell's row lies in the chunk of ordinal bi / 128; cur_chunk holds the last computed row's (i - 1)
            int ch = cur_chunk;
            int o = (i > 0 ? i - 1 : 0) / RK_CHUNK_ROWS;
            while (ch >= 0 && o > bi / RK_CHUNK_ROWS) { ch = __ldcg(p.chunk_prev + ch); o--; }
            bool ops_ok = true;
            __threadfence_block();
            if (!row_walk(p, sh.opsbuf, bi, bj, ch, lane, out.ops_seg, out.n_ops, ops_ok)) out.status |= SFE_ST_INTERNAL;
            if (!ops_ok) out.status |= SFE_ST_OPS_OVERFLOW;
        }
        if (TB) {
            __threadfence();
            __syncwarp();
            int cc = pend_chunk >= 0 ? pend_chunk : cur_chunk;          // (a chunk popped ahead is linked in front of the current one)
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
            if (wide) atomicAdd(&p.counters[CNT_WIDE], 1ULL);
            atomicAdd(&p.counters[CNT_BLOCK_HALVES], 1ULL);
        }
    }
}

// Persistent CTAs.  row_all 1 / 0 / 3: each pulls the next half from a fixed list (every ticket / the first CNT_ROW_N tickets,
// the longest: sfe_launch_tickets' order / the leftovers of the hand-off queue).
// row_all 2: the CTAs SERVE THE HAND-OFF QUEUE while the systolic kernel runs beside them (sfe_launch_ydrop).  An idle CTA
// announces itself (CNT_ROW_FREE++), draws the next queue position and sleeps until that entry is written; a systolic warp
// whose half is still alive at a check-point takes one idle CTA (CNT_ROW_FREE--) and writes exactly one entry, so every entry
// has a CTA waiting for it.  The CTA leaves when every systolic warp has left and its entry is still empty.  The wait is
// bounded (a systolic kernel that never started must not hang the GPU): a CTA that gives up withdraws its announcement, and
// the launcher's leftover pass re-runs whatever was queued but not served.
template <bool TB>
__global__ void __maxnreg__(112) ydrop_row_kernel(const YdParams p)   // 112: one CTA + two systolic blocks fill an SM's registers exactly
{
    __shared__ long long tk_s;
    unsigned smid;
    asm("mov.u32 %0, %%smid;" : "=r"(smid));
    // beside the systolic kernel: tell its start gate that this CTA is resident (sfe_launch_ydrop)
    if ((p.row_all == 0 || p.row_all == 2) && threadIdx.x == 0) atomicAdd(&p.counters[CNT_ROW_STARTED], 1ULL);
    if (p.row_all == 2) {
        for (;;) {
            if (threadIdx.x == 0) {
                atomicAdd(&p.counters[CNT_ROW_FREE], 1ULL);
                const unsigned long long idx = atomicAdd(&p.counters[CNT_LONG_TICKET], 1ULL);
                volatile int32_t *slot = p.long_tickets + idx;
                int t = -1;
                for (long long spin = 0; spin < (1LL << 24); spin++) {           // ~ 1 minute at most
                    t = *slot;
                    if (t >= 0) break;
                    if ((long long)*((volatile unsigned long long *)&p.counters[CNT_SYS_DONE]) >= (long long)p.sys_warps) {
                        __threadfence();
                        t = *slot;                                              // pushed just before the last warp left?
                        break;
                    }
                    __nanosleep(4000);
                }
                if (t < 0) atomicAdd(&p.counters[CNT_ROW_FREE], ~0ULL);          // withdraw (a late claim is caught by the leftover pass)
                tk_s = t;
            }
            __syncthreads();
            const int hid = (int)tk_s;
            __syncthreads();
            if (hid < 0) break;
            __threadfence();                                                    // (the systolic warp's result and returned chunks)
            if (threadIdx.x == 0) atomicAdd(&p.counters[CNT_ROW_BUSY + (smid & 255u)], 1ULL);      // the SM is mine while I work
            row_half<TB>(p, hid);
            __syncthreads();
            if (threadIdx.x == 0) atomicAdd(&p.counters[CNT_ROW_BUSY + (smid & 255u)], ~0ULL);
        }
        return;
    }
    const long long n_row = p.row_all == 1 ? p.n_tickets : (long long)*((volatile unsigned long long *)&p.counters[p.row_all == 3 ? CNT_LONG_LEFT : CNT_ROW_N]);
    const int32_t *tickets = p.row_all == 3 ? p.long_tickets + p.n_tickets : p.tickets;
    for (;;) {
        if (threadIdx.x == 0) tk_s = (long long)atomicAdd(&p.counters[CNT_ROW_TICKET], 1ULL);
        __syncthreads();
        const long long tk = tk_s;
        __syncthreads();
        if (tk >= n_row) break;
        // beside the systolic kernel (row_split) the CTA claims its SM while it works: a half on this kernel is one serial
        // chain of rows, and every other warp on the SM's schedulers stretches it (the systolic warps there sleep meanwhile)
        if (p.row_all == 0 && threadIdx.x == 0) atomicAdd(&p.counters[CNT_ROW_BUSY + (smid & 255u)], 1ULL);
        row_half<TB>(p, tickets[tk]);
        __syncthreads();
        if (p.row_all == 0 && threadIdx.x == 0) atomicAdd(&p.counters[CNT_ROW_BUSY + (smid & 255u)], ~0ULL);
    }
}

// Hand-offs that were queued but not served (a serving CTA gave up, or the systolic kernel outlived them): normally none.
__global__ void select_long_left_kernel(const YdParams p)
{
    const long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    const long long n = (long long)*((volatile unsigned long long *)&p.counters[CNT_LONG_N]);
    if (x >= n) return;
    const int hid = p.long_tickets[x];
    if (hid >= 0 && (p.halves[hid].status & SFE_ST_LONG_PENDING))
        p.long_tickets[p.n_tickets + (long long)atomicAdd(&p.counters[CNT_LONG_LEFT], 1ULL)] = hid;
}

int sfe_launch_long_left(const YdParams &p_in, bool want_tb, int n_sm, cudaStream_t st)
{
    YdParams p = p_in;
    p.row_all = 3; p.row_split = 0;
    const int bs = 256;
    SFE_KL select_long_left_kernel<<<(unsigned)((p.n_tickets + bs - 1) / bs), bs, 0, st>>>(p);
    if (want_tb) SFE_KL ydrop_row_kernel<true><<<(unsigned)n_sm, RK_THREADS, 0, st>>>(p);
    else SFE_KL ydrop_row_kernel<false><<<(unsigned)n_sm, RK_THREADS, 0, st>>>(p);
    SFE_LAUNCH_CHECK();
}

int sfe_launch_ydrop_row(const YdParams &p, bool want_tb, long long grid, cudaStream_t st)
{
    if (grid < 1) grid = 1;
    if (want_tb) SFE_KL ydrop_row_kernel<true><<<(unsigned)grid, RK_THREADS, 0, st>>>(p);
    else SFE_KL ydrop_row_kernel<false><<<(unsigned)grid, RK_THREADS, 0, st>>>(p);
    SFE_LAUNCH_CHECK();
}
