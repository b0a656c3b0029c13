// ydrop_kernel.cu -- the warp-systolic Y-drop gapped extension.
//
// One warp = one one-sided extension ("anchor-half").  The paper's kernel
// (Fig. 8) gives each thread one line of the DP matrix and passes neighbour values
// between threads; this kernel keeps that systolic idea but is organised for sm_100a:
//   * rows are processed in strips of 32 (lane l owns row 32 s + l), each lane sweeping its row
//     left to right SK columns behind the lane above (SK = 1, or 2 for the longest tickets), so that
//     32 lanes stay busy whatever the width of the live band is (0..~700 columns, changing every row);
//   * per cell: PRMT score lookup from a packed int8 row, IADD3, two VIADDMNMX (E, F), one
//     VIMNMX3 (H) -- the Blackwell DPX instructions -- plus compare/select for the Y-drop prune;
//   * lane-to-lane messages and the strip-to-strip boundary row go through a 10 KiB per-warp
//     shared-memory area laid out so that every access of the 16x unrolled loop is base+immediate;
//   * 4 traceback bits per cell are packed 8 cells to a word and written as one coalesced 256 B
//     record per warp per 16 steps into the recycled HBM arena (R11);
//   * rows are pruned with the row-lagged threshold T(r) = best(rows <= r - 32) - ydrop (R4),
//     which is exactly what is final when row r starts in this schedule;
//   * when the half is done the same warp walks its traceback (walk_traceback: 32 path cells per
//     ballot), stages the run-length ops and gives its chunks back to the free ring (a8).
// Dead cells are gated only on the diagonal/open edge (R6 lemma).
#include "sfe_internal.cuh"
#include "ydrop_common.cuh"

#ifndef SFE_LONG_SKEW
#define SFE_LONG_SKEW 2           // lane skew used for the reserved (longest) tickets; 1 = same as the others
#endif
#ifndef SFE_MIN_BLOCKS
#define SFE_MIN_BLOCKS 3
#endif
#ifndef SFE_BLOCK_THREADS
#define SFE_BLOCK_THREADS 192     // 6 warps x 12.3 KB of shared memory; 3 blocks = 18 warps per SM
#endif
// Ordering of a lane's message store and the next lane's load of it inside one wavefront step.
#define SFE_STEP_FENCE() __syncwarp()

// Boundary-ring address of column c: row (c-1) mod 8, segment ((c-1) div 8) mod RING/8.  Strips start
// at a multiple of 16 and groups hold 16 steps, so lane 0 (reading column cs+t0+k+1) and lane 31
// (writing column cs+t0+k-31) both touch row k&7 and segment base + (k>>3) with an EVEN base: no
// ring wrap inside a group, every access of the unrolled loop is base + immediate.
template <int RL2, int SK>
static __device__ __forceinline__ int bnd_off(int c)
{
    const int u = c - SK;
    return (u & 7) * RingGeom<RL2>::ROW_STRIDE + SFE_EXCH_BYTES + ((u >> 3) & (RingGeom<RL2>::RING / 8 - 1)) * 8;
}

// fill selector-ring entries for columns [lo, hi).  Common case (every column has a target base): each
// lane takes one byte of the 2-bit plane = 4 bases, plus their 4 mask bits -- two loads per 4 columns.
template <int RL2>
static __device__ __forceinline__ void fill_sel(uint16_t *selring, const HalfGeom &g, int lo, int hi, int lane)
{
    typedef RingGeom<RL2> G;
    if (lo <= 0 || hi - 1 > g.m) {                          // strip start / right edge of the DP matrix: per column
        for (int c = lo + lane; c < hi; c += 32) {
            const uint16_t v = (uint16_t)col_selector(g, c);
            const int idx = c & (G::SELRING - 1);
            selring[idx] = v;
            if (idx < 32) selring[idx + G::SELRING] = v;
        }
    } else {
        const long long ka = g.t0 + (long long)g.d * lo, kb = g.t0 + (long long)g.d * (hi - 1);
        const long long kmin = ka < kb ? ka : kb, kmax = ka < kb ? kb : ka;
        for (long long B = (kmin >> 2) + lane; B <= (kmax >> 2); B += 32) {
            const uint32_t cb = g.tc[B];
            const uint32_t mb = (uint32_t)g.tm[B >> 1] >> ((B & 1) * 4);
#pragma unroll
            for (int e = 0; e < 4; e++) {
                const int c = g.d * (int)(4 * B + e - g.t0);
                if (c >= lo && c < hi) {
                    const uint32_t code = (cb >> (2 * e)) & 3u;
                    const uint16_t v = (uint16_t)(((mb >> e) & 1u) ? 0xCCC4u : 0x8880u + 0x1111u * code);
                    const int idx = c & (G::SELRING - 1);
                    selring[idx] = v;
                    if (idx < 32) selring[idx + G::SELRING] = v;
                }
            }
        }
    }
    __syncwarp();
}

// fill boundary-ring entries for columns [lo, hi) with "dead"
template <int RL2, int SK>
static __device__ __forceinline__ void fill_bnd_neg(char *wbase, int lo, int hi, int lane)
{
    for (int c = lo + lane; c < hi; c += 32) *(int2 *)(wbase + bnd_off<RL2, SK>(c)) = make_int2(SFE_NEG, SFE_NEG);
    __syncwarp();
}

struct TbWriter {
    uint32_t *pool; int32_t *chunk_prev; int32_t *ring; SfeFreeRing *ring_state; int n_chunks;
    uint32_t *ptr;          // this lane's word pair of the next record
    int left;               // records left in the current chunk
    int cur_chunk; int nrec; bool ok;
    __device__ __forceinline__ void put(uint32_t w0, uint32_t w1, int lane)
    {
        if (!ok) return;
        if (left == 0) {
            const int c = chunk_pop(ring, ring_state, n_chunks, lane);
            if (c < 0) { ok = false; left = c == -2 ? -1 : 0; return; }      // left == -1 remembers an abandoned wait (counted at the end)
            if (lane == 0) chunk_prev[c] = cur_chunk;
            cur_chunk = c;
            ptr = pool + (size_t)c * SFE_CHUNK_RECS * SFE_REC_WORDS + 2 * lane;
            left = SFE_CHUNK_RECS;
        }
        *(uint2 *)ptr = make_uint2(w0, w1);
        ptr += SFE_REC_WORDS; left--; nrec++;
    }
    // give every chunk of this half back (after the walk, or when the half is abandoned)
    __device__ __forceinline__ void release(int lane, unsigned long long *counters)
    {
        // One fence per half: this warp's record stores must have landed before a chunk changes owner.
        // (A gpu-scope fence also invalidates the SM's L1, so it is not done per chunk.)
        __threadfence();
        __syncwarp();
        int c = cur_chunk;
        while (c >= 0) {
            const int prev = __ldcg(chunk_prev + c);        // same address in every lane
            chunk_push(ring, ring_state, n_chunks, c, counters + CNT_RING_DROPS, lane);
            c = prev;
        }
        cur_chunk = -1;
    }
};

// Integer subtraction on the FMA pipe (IMAD), which the ALU-heavy hot loop leaves mostly idle.
static __device__ __forceinline__ int fma_sub(int a, int b)      // a - b
{
    int r;
    asm("mad.lo.s32 %0, %1, -1, %2;" : "=r"(r) : "r"(b), "r"(a));
    return r;
}
// acc = (acc << 1) | (sign bit of x): one SHF.L.W
static __device__ __forceinline__ uint32_t shift_in_sign(uint32_t acc, int x) { return __funnelshift_l((uint32_t)x, acc, 1); }

// One group of 16 wavefront steps.  Everything indexed by k is an immediate after unrolling.
// Per cell: LDS.U16 + PRMT (score), IADD3 (M), 2 x VIADDMNMX (E, F), VIMNMX3 (H), compare + select
// (alive gate, R5/R6), 4 x (subtract + funnel shift) for the traceback nibble, half a VIMNMX3 (best), and
// the message STS.64 / LDS.64.  The kernel is issue-bound (profiles/r1_02), so what counts is the
// number of instructions, not the pipe they run on; the subtractions stay on the FMA pipe (IMAD).
// Traceback: four bit PLANES per lane per group, step k at bit 15-k of each (acc0 = plane3 << 16 | plane2 ... see below):
//   plane 3 = H not from M, plane 2 = H not from E, plane 1 = E extended, plane 0 = F extended (R11).
// One accumulator per plane: four independent shift chains of one SHF per step instead of one chain of four (the
// pointer bits of a long half are a second loop-carried dependency next to the DP's own).
// dead: bit 15-k set iff the cell of step k is dead.
// The position of a new lane-local best (strict '>', R7) is found after the group, only by the
// lanes whose best rose: the first k with H_k == best is the last strict increase.
// SK = lane skew in columns.  SK = 1: lane l is one column behind lane l-1 (fewest idle steps per strip).
// SK = 2: two columns behind, so the message loaded in step k is consumed in step k+2 and its LDS latency
// leaves the per-step dependency chain: a shorter step for the halves whose serial chain bounds the run.
template <bool TB, bool EDGE, int RL2, bool GLOBAL, int SK>
static __device__ __forceinline__ void run_group16(int &upH, int &upE, int2 &pend, uint32_t &sel_nx, int &dg, int &F, int &Hgl, int &best, int &best_t,
                                                   uint32_t &acc0, uint32_t &acc1, uint32_t &dead, const uint32_t srow_lo,
                                                   const uint32_t srow_hi, const int T, const int OX, const int X,
                                                   const char *rptr, char *wptr, const uint16_t *selp, const int col0,
                                                   const int m, const int t0)
{
#ifdef SFE_SHFL_HANDOFF
    const bool lane_is0 = sfe_lane() == 0, lane_is31 = sfe_lane() == 31;
#endif
    typedef RingGeom<RL2> G;
    const int best_in = best;
    uint32_t pl3 = 0, pl2 = 0, pl1 = 0, pl0 = 0;
    int Hk[16];
#pragma unroll
    for (int k = 0; k < 16; k++) {
        const int off = (k & 7) * G::ROW_STRIDE + (k >> 3) * 8;
        const uint32_t sel = sel_nx;                       // loaded a whole step ahead: off the critical path
        sel_nx = GLOBAL ? __ldcg(selp + k + 1) : selp[k + 1];
        const int s = prmt_sx(srow_lo, srow_hi, sel);
        const int M = dg + s + OX;                         // dg = H(i-1,j-1) - OX, or NEG if dead
        const int E = __viaddmax_s32(upE, -X, upH);        // upH = H(i-1,j) - OX, or NEG if dead
        const int Fn = __viaddmax_s32(F, -X, Hgl);         // Hgl = H(i,j-1) - OX (ungated: R6 lemma)
        int H = __vimax3_s32(M, E, Fn);
        if (EDGE) { if (col0 + k > m) H = SFE_NEG; }       // beyond the target end
        Hk[k] = H;
        const bool isdead = H < T;                         // R5: alive <=> H >= T
        const int Hg = H - OX;
        if (TB) {
            pl3 = shift_in_sign(pl3, fma_sub(M, H));       // M < H  <=> H not from M
            pl2 = shift_in_sign(pl2, fma_sub(E, H));       // E < H  <=> H not from E
            pl1 = shift_in_sign(pl1, fma_sub(upH, E));     // upH < E <=> E extended (open wins ties)
            pl0 = shift_in_sign(pl0, fma_sub(Hgl, Fn));    // Hgl < F <=> F extended
        }
        if (isdead) dead |= 0x8000u >> k;
        if (k & 1) best = __vimax3_s32(best, Hk[k - 1], H); // one VIMNMX3 per two cells
        const int msgH = isdead ? SFE_NEG : Hg;            // dead cells send NEG on the diagonal / open edge
#ifdef SFE_SHFL_HANDOFF
        // A/B variant ("previous thread's values ... via warp shuffle"): lanes 1..31 take the message from the
        // lane above by shuffle; shared memory only carries the strip-to-strip boundary row (lane 31 writes, lane 0 reads).
        // Measured slower than the shared-memory exchange on sm_100a (profiles/r2_05): two SHFL per step replace one
        // STS.64 + LDS.64 pair on the same MIO path and their latency sits on the step's dependency chain.
        if (lane_is31) *(int2 *)(wptr + off) = make_int2(msgH, E);
        dg = upH; F = Fn; Hgl = Hg;
        int2 u;
        u.x = __shfl_up_sync(FULL, msgH, 1); u.y = __shfl_up_sync(FULL, E, 1);
        if (lane_is0) u = GLOBAL ? __ldcg((const int2 *)(rptr + off)) : *(const int2 *)(rptr + off);
#else
        *(int2 *)(wptr + off) = make_int2(msgH, E);
        dg = upH; F = Fn; Hgl = Hg;
        SFE_STEP_FENCE();
        const int2 u = GLOBAL ? __ldcg((const int2 *)(rptr + off)) : *(const int2 *)(rptr + off);
#endif
        if (SK == 1) { upH = u.x; upE = u.y; }             // the lane above is one column ahead: used in the next step
        else { upH = pend.x; upE = pend.y; pend = u; }     // two columns ahead: used the step after next
    }
    if (TB) { acc0 = __byte_perm(pl2, pl3, 0x5410); acc1 = __byte_perm(pl0, pl1, 0x5410); }   // plane3:plane2, plane1:plane0
    if (best > best_in) {
        int kk = 15;
#pragma unroll
        for (int k = 14; k >= 0; k--) kk = Hk[k] == best ? k : kk;
        best_t = t0 + kk;
    }
}

// ---- a8, first part: warp-cooperative traceback walk ---------------------------------------------
// Runs in the warp that has just finished the half, while its records are the most recently
// written lines of the arena.  Control flow is uniform: every lane holds the same (i, j, state).
// A window of SFE_WALK_WIN_RECS records of the current strip is copied to shared memory (each lane
// loads its own 8 bytes of every record: coalesced); then up to 32 consecutive path cells are
// examined at once -- lane k looks at the k-th cell in the current direction (diagonal for state
// H, up for E, left for F, R11) -- and a ballot finds where the run stops.
struct TbReader {                       // random access to this half's records; all lanes hold the same cursor
    const uint32_t *pool; const int32_t *chunk_prev;
    int chunk, ord, last_chunk, last_ord, nrec;
    int up_chunk, up_ord;               // the chunk one above the cursor (ordinal ord + 1), -1 if not known
    bool bad;                           // an index outside the half's records was asked for (never expected)
    __device__ __forceinline__ const uint32_t *rec(int ridx)
    {
        if (ridx < 0 || ridx >= nrec) { bad = true; ridx = 0; }
        const int o = ridx / SFE_CHUNK_RECS;
        // The walk visits records in (mostly) decreasing order, but a strip's header may sit in the chunk below the
        // strip's records: going back UP one chunk must not restart from the end of the chain (a half of 5 * 10^5 rows has
        // ~300 chunks: that restart cost 28,000 cycles per strip, a third of the whole traceback pass, until round 2).
        if (o > ord) {
            if (o == up_ord && up_chunk >= 0) { chunk = up_chunk; ord = up_ord; up_chunk = -1; }
            else { chunk = last_chunk; ord = last_ord; up_chunk = -1; }
        }
        while (ord > o) { up_chunk = chunk; up_ord = ord; chunk = __ldcg(chunk_prev + chunk); ord--; }
        return pool + ((size_t)chunk * SFE_CHUNK_RECS + (ridx - o * SFE_CHUNK_RECS)) * SFE_REC_WORDS;
    }
};

// Returns false if the walk did not reach the origin (internal error guard).
template <int SK>
static __device__ bool walk_traceback(const YdParams &p, TbReader &rd, const int end_i, const int end_j, int hdr, int strip,
                                      char *wk, const int lane, uint32_t &ops_seg, int &n_ops, bool &ops_ok)
{
    uint32_t *win = (uint32_t *)wk;
    OpsWriter ow;
    ow.buf = (uint32_t *)(wk + SFE_WALK_WIN_RECS * SFE_REC_BYTES);
    ow.stage = p.ops_stage; ow.used = &p.counters[CNT_OPS]; ow.cap = p.ops_cap;
    ow.nbuf = 0; ow.nops = 0; ow.cur_op = -1; ow.run = 0; ow.prev_seg = SFE_NO_SEG; ow.ok = true;
    ops_seg = SFE_NO_SEG; n_ops = 0; ops_ok = true;
    if (end_i == 0 && end_j == 0) return true;
    __syncwarp();                                        // the records of this half, written lane by lane, are visible
    int i = end_i, j = end_j, state = 0;
    const uint32_t *hr = rd.rec(hdr);
    uint2 hv = __ldcg((const uint2 *)hr);
    int cs = (int)hv.x, prev_hdr = (int)hv.y;
    while (strip > (i >> 5)) { hdr = prev_hdr; strip--; hr = rd.rec(hdr); hv = __ldcg((const uint2 *)hr); cs = (int)hv.x; prev_hdr = (int)hv.y; }
    int win_lo = 0, win_hi = -1;                         // record groups of this strip held in win[]
    int pre_idx = -1; uint2 pre_hv = make_uint2(0u, 0u); // header of the strip above, loaded ahead
    long long guard = 3LL * ((long long)end_i + end_j) + 4LL * (strip + 1) + 64;
    while (!(i == 0 && j == 0 && state == 0)) {
        if (--guard < 0 || rd.bad) return false;
        if ((i >> 5) < strip) {                          // crossed into the strip above
            hdr = prev_hdr; strip--;
            if (pre_idx == hdr) hv = pre_hv; else { hr = rd.rec(hdr); hv = __ldcg((const uint2 *)hr); }
            cs = (int)hv.x; prev_hdr = (int)hv.y;
            win_hi = -1;
        }
        const int L = i & 31;
        const int t = j - cs + SK * L;                   // step of cell (i, j) in its strip
        const int g = t >> 4;
        if (g > win_hi || g < win_lo) {                  // (re)load the window: groups g-7 .. g
            __syncwarp();
            win_hi = g; win_lo = max(0, g - (SFE_WALK_WIN_RECS - 1));
            // The window's records are consecutive and span at most two chunks: resolve the two chunk bases first, then the
            // loads are plain address arithmetic and independent of one another -- one memory latency per window, not one
            // per record (the records of a long half were written long ago: they come from HBM, ~800 cycles each).
            const int r_hi = hdr + 1 + win_hi, r_lo = hdr + 1 + win_lo;
            const int o_hi = r_hi / SFE_CHUNK_RECS;
            const uint32_t *b_hi = rd.rec(r_hi) - (size_t)(r_hi - o_hi * SFE_CHUNK_RECS) * SFE_REC_WORDS;
            const uint32_t *b_lo = rd.rec(r_lo) - (size_t)(r_lo - (r_lo / SFE_CHUNK_RECS) * SFE_CHUNK_RECS) * SFE_REC_WORDS;
            if (prev_hdr >= 0 && pre_idx != prev_hdr) { pre_idx = prev_hdr; pre_hv = __ldcg((const uint2 *)rd.rec(prev_hdr)); }   // next strip's header, early
            uint2 wv[SFE_WALK_WIN_RECS];
#pragma unroll
            for (int y = 0; y < SFE_WALK_WIN_RECS; y++) {
                const int r = r_lo + y;
                const int o = r / SFE_CHUNK_RECS;
                const uint32_t *src = (o == o_hi ? b_hi : b_lo) + (size_t)(r - o * SFE_CHUNK_RECS) * SFE_REC_WORDS + 2 * lane;
                wv[y] = r <= r_hi ? __ldcg((const uint2 *)src) : make_uint2(0u, 0u);
            }
#pragma unroll
            for (int y = 0; y < SFE_WALK_WIN_RECS; y++) *(uint2 *)(win + y * SFE_REC_WORDS + 2 * lane) = wv[y];
            __syncwarp();
        }
        // lane k examines the k-th cell from (i, j) in the direction of the current state
        const int di = state == 2 ? 0 : 1, dj = state == 1 ? 0 : 1;
        const int Lk = L - lane * di;
        const int tk = t - lane * (SK * di + dj);
        const bool valid = Lk >= 0 && tk >= 0 && (tk >> 4) >= win_lo;
        uint32_t nib = 0;
        if (valid) {
            const uint2 w = *(const uint2 *)(win + ((tk >> 4) - win_lo) * SFE_REC_WORDS + 2 * Lk);    // planes 3:2, 1:0 of that lane and group
            const int sft = 15 - (tk & 15);
            nib = (((w.x >> (16 + sft)) & 1u) << 3) | (((w.x >> sft) & 1u) << 2) | (((w.y >> (16 + sft)) & 1u) << 1) | ((w.y >> sft) & 1u);
        }
        // nib: bit3 = H not from M, bit2 = H not from E, bit1 = E extended, bit0 = F extended
        const bool cont = state == 0 ? !(nib & 8u) : (state == 1 ? (nib & 2u) != 0 : (nib & 1u) != 0);
        const bool origin = i == lane * di && j == lane * dj;   // the walk ends at (0,0), whose own nibble says "from M"
        const uint32_t stop = __ballot_sync(FULL, !(valid && cont) || origin);
        const uint32_t vmask = __ballot_sync(FULL, valid);
        const int pstop = stop ? __ffs(stop) - 1 : 32;   // cells 0 .. pstop-1 continue the run
        const bool stop_valid = pstop < 32 && ((vmask >> pstop) & 1u);
        if (state == 0) {
            ow.emit(SFE_OP_M, pstop, lane);
            i -= pstop; j -= pstop;
            if (stop_valid && !(i == 0 && j == 0)) {     // cell pstop is not from M: switch to its gap state, same cell
                const uint32_t nb = __shfl_sync(FULL, nib, pstop);
                state = (nb & 4u) ? 2 : 1;
            }
        } else if (state == 1) {                         // E: every visited cell emits I; the cell that opened returns to H
            const int cnt = stop_valid ? pstop + 1 : pstop;
            ow.emit(SFE_OP_I, cnt, lane);
            i -= cnt;
            if (stop_valid) state = 0;
        } else {                                         // F likewise with D
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

// A check-point of a long half: take one of the idle row-kernel CTAs if the rule allows it.  A hand-off restarts the half, so
// it pays only early in the half's life: there are four check-points (long_strips x 1, 2, 4, 8 strips; a restart at the last
// one costs 8 long_strips strips of the row kernel at most if the half was about to end).  The early ones leave a reserve for
// halves with more evidence of being long: more than 3/4, 1/2, 1/4 of the CTAs must be idle, the last one takes any.
// Every successful claim is matched by exactly one push to the hand-off queue.
static __device__ __forceinline__ bool claim_row_cta(unsigned long long *counters, int slots, int level, int lane)
{
    int got = 0;
    if (lane == 0) {
        const long long reserve = level >= 3 ? 0 : (long long)slots * (3 - level) / 4;
        if ((long long)*((volatile unsigned long long *)&counters[CNT_ROW_FREE]) > reserve) {
            const long long f = (long long)atomicAdd(&counters[CNT_ROW_FREE], ~0ULL);       // FREE--, returns the old value
            if (f > reserve) got = 1;
            else atomicAdd(&counters[CNT_ROW_FREE], 1ULL);
        }
    }
    return __shfl_sync(FULL, got, 0) != 0;
}

template <bool TB, int RL2, bool GLOBAL, int SK, bool COOP = false>
// COOP: the variant with the hand-off check-points (a second instantiation: the plain one's code must not carry them,
// C4 was 3 % slower with them compiled in).
// Returns false only when SK == 2 and a strip outgrew the shared-memory window (skew 2 needs 31 more steps per strip):
// nothing has been published then, and the caller runs the half again with SK == 1.
static __device__ bool extend_half(const YdParams &p, const int hid, char *wsm, char *wk, const int lane, const uint32_t mode_bits)
{
    typedef RingGeom<RL2> G;
    uint16_t *selring = (uint16_t *)(wsm + 8 * G::ROW_STRIDE);
    sfe_half out;
    out.score = 0; out.end_i = 0; out.end_j = 0; out.status = 0; out.cells = 0;
    out.ops_seg = SFE_NO_SEG; out.n_ops = 0; out.n_strips = 0; out.n_rec = 0; out.steps = 0; out.max_steps = 0;
    out.cycles = 0; out.smid = 0; out.wslot = 0;
    const long long clk0 = clock64();

    HalfGeom g;
    if (!half_setup(p, hid, g)) {
        out.status = SFE_ST_BAD_ANCHOR;
        if (lane == 0) p.halves[hid] = out;
        return true;
    }

    const int OX = p.OX, X = p.X;
    TbWriter tb;
    tb.pool = p.pool; tb.chunk_prev = p.chunk_prev; tb.ring = p.free_ring; tb.ring_state = p.ring_state; tb.n_chunks = p.n_chunks;
    tb.cur_chunk = -1; tb.nrec = 0; tb.ok = TB; tb.ptr = nullptr; tb.left = 0;

    int best = 0, best_i = 0, best_j = 0;     // lane-local first maximum
    int cumA = 0, cumB = 0;                    // lane-local best through the previous strip / the one before
    unsigned long long cells = 0;
    int cs = 0, prevR = -1;
    int bnd_valid = 0;                         // boundary ring holds row (r0-1) for columns < bnd_valid
    int sel_hi = -32 * SK;                     // selector ring is filled for columns < sel_hi (lane 31 starts at column -31 SK)
    int total_steps = 0, max_steps = 0, last_hdr = -1, n_strips = 0;
    bool wide = false, limit = false, lng = false;
    // hand-off: a half still alive at a check-point (long_strips, 2 long_strips, 4 long_strips ... strips) is one of the pass's
    // long serial chains.  If a CTA of the cooperative row kernel is idle it stops here, queues itself, and that CTA re-runs it
    // from its start: a row costs the CTA a third less, and it has its SM to itself (ydrop_row_kernel.cu, sfe_launch_ydrop).
    // (long_strips is a power of two, so the check-points are the powers of two >= it: no state is carried through the loop)

    for (int s = 0;; s++) {
        const int r0 = s * 32;
        if (r0 > g.n) break;
        if (COOP && !GLOBAL && s >= p.long_strips && (s & (s - 1)) == 0 && p.long_strips > 0 && s <= 8 * p.long_strips) {
            if (claim_row_cta(p.counters, p.row_slots, __clz(p.long_strips) - __clz(s), lane)) { lng = true; break; }
        }
        const int r = r0 + lane;
        const bool active = r <= g.n;
        // R4: T(r) = best over rows <= r - 32, minus ydrop.  Rows <= r - 32 are: every row of
        // strips <= s-2 (cumB of all lanes) and the rows of strip s-1 held by lanes <= lane.
        int pm = cumA;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(FULL, pm, o); if (lane >= o) pm = max(pm, v); }
        int ab = cumB;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) ab = max(ab, __shfl_xor_sync(FULL, ab, o));
        const int B = max(pm, ab);
        const int T = !active ? (1 << 29) : (p.ydrop_inf ? SFE_T_INF : B - p.Y);   // rows beyond the query: never alive (scores < 2^29, R25)
        uint32_t srow_lo;
        if (!active) srow_lo = 0x80808080u;
        else if (r == 0) srow_lo = 0u;
        else srow_lo = p.srow[sfe_base(g.qc, g.qm, g.q0 + (long long)g.d * r)];
        const uint32_t srow_hi = p.srow_hi;

        if (TB) {   // strip header record: lane 0's word pair = (cs, previous header's record index)
            const int hdr = tb.nrec;
            tb.put(lane == 0 ? (uint32_t)cs : (uint32_t)s, lane == 0 ? (uint32_t)last_hdr : 0u, lane);
            last_hdr = hdr;
        }
        n_strips++;

        if (sel_hi < cs - 32 * SK) sel_hi = cs - 32 * SK;
        if (bnd_valid <= cs + SK - 1) { fill_bnd_neg<RL2, SK>(wsm, bnd_valid, cs + 64, lane); bnd_valid = cs + 64; }
        int refill_at = min(sel_hi - 1, bnd_valid - SK);     // first cmax that needs a ring refill (the selector of column cmax+1 is prefetched)
        int upH = SFE_NEG, upE = SFE_NEG, dg = SFE_NEG, F = SFE_NEG, Hgl = SFE_NEG;
        int2 pend = make_int2(SFE_NEG, SFE_NEG);
        if (lane == 0) {
            const int2 u = GLOBAL ? __ldcg((const int2 *)(wsm + bnd_off<RL2, SK>(cs))) : *(const int2 *)(wsm + bnd_off<RL2, SK>(cs));
            upH = u.x; upE = u.y;
            if (SK == 2) pend = GLOBAL ? __ldcg((const int2 *)(wsm + bnd_off<RL2, SK>(cs + 1))) : *(const int2 *)(wsm + bnd_off<RL2, SK>(cs + 1));
            if (s == 0) dg = -OX;                           // R8: H(0,0) = 0 enters as the diagonal of (0,0)
        }
        // alive bits (step k of the group at bit 15-k) of the first / last group of my row that had an alive cell
        uint32_t first_al = 0, last_al = 0;
        int first_g = 0, last_g = 0, best_t = -1;
        const int best_before = best;
        int t0 = 0;
        bool bail = false;
        // Message pointers.  Lanes 1..31 read the exchange slot of the lane above and lanes 0..30 write
        // their own (fixed addresses); lane 0 reads and lane 31 writes the boundary ring, whose byte
        // offset advances by 16 (two segments) per group.
        const bool is0 = lane == 0, is31 = lane == 31;
        char *const bnd = wsm + SFE_EXCH_BYTES;
        const char *const rbase = is0 ? bnd : wsm + (lane - 1) * 8;           // (exchange slots do not depend on the skew)
        char *const wbase = is31 ? bnd : wsm + lane * 8;
        const int rstride = is0 ? 16 : 0, wstride = is31 ? 16 : 0;
        int roff = is0 ? (cs & (G::RING - 1)) : 0;           // column cs+t0+k+1 -> segment (cs+t0)/8 + (k>>3)
        int woff = is31 ? ((cs - 32 * SK) & (G::RING - 1)) : 0;   // column cs+t0+k-31 SK -> segment (cs+t0-32 SK)/8 + (k>>3)
        for (;; t0 += 16) {
            const int cmax = cs + t0 + 15;                  // lane 0's last column of this group
            if (cmax >= refill_at) {
                if (sel_hi <= cmax + 1) { fill_sel<RL2>(selring, g, sel_hi, cmax + 129, lane); sel_hi = cmax + 129; }
                if (bnd_valid <= cmax + SK) { fill_bnd_neg<RL2, SK>(wsm, bnd_valid, bnd_valid + 64, lane); bnd_valid += 64; }
                refill_at = min(sel_hi - 1, bnd_valid - SK);
            }
            const char *rptr = rbase + roff;
            char *wptr = wbase + woff;
            roff = (roff + rstride) & (G::RING - 1);
            woff = (woff + wstride) & (G::RING - 1);
            const int col0 = cs + t0 - SK * lane;
            const uint16_t *selp = selring + (col0 & (G::SELRING - 1));
            uint32_t sel_nx = GLOBAL ? __ldcg(selp) : selp[0];
            uint32_t acc0 = 0, acc1 = 0, dead = 0;
            if (cmax > g.m)
                run_group16<TB, true, RL2, GLOBAL, SK>(upH, upE, pend, sel_nx, dg, F, Hgl, best, best_t, acc0, acc1, dead, srow_lo, srow_hi, T, OX, X,
                                                   rptr, wptr, selp, col0, g.m, t0);
            else
                run_group16<TB, false, RL2, GLOBAL, SK>(upH, upE, pend, sel_nx, dg, F, Hgl, best, best_t, acc0, acc1, dead, srow_lo, srow_hi, T, OX, X,
                                                    rptr, wptr, selp, col0, g.m, t0);
            if (TB) tb.put(acc0, acc1, lane);
            const uint32_t al = ~dead & 0xffffu;
            if (al) {
                if (!first_al) { first_al = al; first_g = t0; }
                last_al = al; last_g = t0;
            }
            // End of the strip.  A cell needs an alive predecessor: left = my previous step, up / diagonal = the lane above
            // SK / SK + 1 steps earlier (lane 0: the boundary row, dead beyond column prevR + 1).  So SK + 1 consecutive steps
            // in which no lane has an alive cell, with lane 0 already past prevR + 1, prove that nothing can come alive any
            // more -- no need to run a whole dead group to find out.  anyal: bit 15 - k = some lane alive in step k.
            const uint32_t anyal = __reduce_or_sync(FULL, al);
            const int tz = __ffs(anyal | 0x10000u) - 1;     // trailing all-dead steps of this group (0 .. 16)
            if (tz >= SK + 1 && cs + t0 + 16 - (SK + 1) > prevR + 1) { t0 += 16; break; }
            if (t0 + 16 >= G::MAX_STEPS - 16 * (SK - 1)) { t0 += 16; bail = true; break; }
        }
        const int first = first_al ? cs - SK * lane + first_g + __clz(first_al) - 16 : 0x7fffffff;
        const int last = last_al ? cs - SK * lane + last_g + 16 - __ffs(last_al) : -1;
        total_steps += t0;
        if (t0 > max_steps) max_steps = t0;
        if (bail) { wide = true; break; }
        if (last >= 0) cells += (unsigned long long)(last - first + 1);
        if (best > best_before) { best_i = r; best_j = cs + best_t - SK * lane; }
        cumB = cumA; cumA = best;
        if (__any_sync(FULL, best >= SFE_SCORE_LIMIT)) { limit = true; break; }   // R25: one test per strip
        const int L31 = __shfl_sync(FULL, first, 31), R31 = __shfl_sync(FULL, last, 31);
        if (R31 < 0) break;                                 // last row of the strip has no alive cell
        bnd_valid = cs + t0 - 31 * SK;                      // lane 31 wrote columns cs-31 SK .. cs+t0-31 SK-1
        prevR = R31;
        cs = L31 & ~15;
    }

    // warp reduction of the lane-local first maxima: key (score desc, i asc, j asc) (R7)
    int bs = best, bi = best_i, bj = best_j;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const int os = __shfl_xor_sync(FULL, bs, o), oi = __shfl_xor_sync(FULL, bi, o), oj = __shfl_xor_sync(FULL, bj, o);
        const bool take = os > bs || (os == bs && (oi < bi || (oi == bi && oj < bj)));
        if (take) { bs = os; bi = oi; bj = oj; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) cells += __shfl_xor_sync(FULL, cells, o);
    if (SK == 2 && wide) {                                  // too wide for the skew-2 schedule: give the chunks back, try again with skew 1
        if (TB) tb.release(lane, p.counters);
        return false;
    }
    // every lane holds the same winner; the broadcast makes that visible to the compiler's uniformity
    // analysis, so that the walk below (and the next half after it) compiles as warp-uniform code
    bs = __shfl_sync(FULL, bs, 0); bi = __shfl_sync(FULL, bi, 0); bj = __shfl_sync(FULL, bj, 0);

    out.score = bs; out.end_i = bi; out.end_j = bj; out.cells = cells;
    // normal kernel: a bail-out is re-run by the wide kernel; wide kernel: a bail-out is final (band limit)
    out.status = (wide ? (GLOBAL ? (SFE_ST_WIDE | SFE_ST_BAND_LIMIT) : SFE_ST_WIDE_PENDING) : (GLOBAL ? SFE_ST_WIDE : 0u)) |
                 ((TB && !tb.ok && !lng) ? SFE_ST_PASS_OVERFLOW : 0u) | (limit ? SFE_ST_SCORE_LIMIT : 0u) | (lng ? SFE_ST_LONG_PENDING : 0u) | mode_bits;
    out.n_strips = n_strips; out.n_rec = tb.nrec;
    if (TB && tb.ok && !wide && !limit && !lng) {                             // a8: walk the pointers now, stage the run-length ops
        TbReader rd;
        rd.pool = p.pool; rd.chunk_prev = p.chunk_prev; rd.chunk = tb.cur_chunk; rd.ord = (tb.nrec - 1) / SFE_CHUNK_RECS;
        rd.last_chunk = rd.chunk; rd.last_ord = rd.ord; rd.nrec = tb.nrec; rd.bad = false; rd.up_chunk = -1; rd.up_ord = -1;
        bool ops_ok = true;
        if (!walk_traceback<SK>(p, rd, bi, bj, last_hdr, n_strips - 1, wk, lane, out.ops_seg, out.n_ops, ops_ok))
            out.status |= SFE_ST_INTERNAL;
        if (!ops_ok) out.status |= SFE_ST_OPS_OVERFLOW;
    }
    if (TB) tb.release(lane, p.counters);
    out.steps = total_steps; out.max_steps = max_steps;
    {   // per-half profile (Fig. 5: per-anchor runtime spread): SM cycles spent, where it ran
        unsigned smid, wslot;
        asm("mov.u32 %0, %%smid;" : "=r"(smid));
        asm("mov.u32 %0, %%warpid;" : "=r"(wslot));
        out.cycles = clock64() - clk0; out.smid = smid; out.wslot = wslot;
    }
    if (lane == 0) {
        p.halves[hid] = out;
        atomicAdd(&p.counters[CNT_STEPS], (unsigned long long)total_steps);
        if (TB) atomicAdd(&p.counters[CNT_TBBYTES], (unsigned long long)tb.nrec * (unsigned long long)SFE_REC_BYTES);
        if (TB && !tb.ok && !lng) atomicAdd(&p.counters[CNT_OVERFLOW], 1ULL);
        if (TB && !tb.ok && tb.left < 0) atomicAdd(&p.counters[CNT_RING_DROPS], 1ULL);
        if (wide && !GLOBAL) atomicAdd(&p.counters[CNT_WIDE], 1ULL);
        if (lng) {                                            // (the result above and the returned chunks are visible before the ticket is)
            __threadfence();
            const unsigned long long pos = atomicAdd(&p.counters[CNT_LONG_N], 1ULL);
            *((volatile int32_t *)&p.long_tickets[pos]) = hid;
        }
    }
    return true;
}

// Persistent kernel: every warp pulls anchor-half tickets from one atomic counter (a3).
// While a row-kernel CTA works on this SM (row_split passes) the systolic warps here take no new ticket: they sleep, the
// other SMs' warps drain the queue, and the CTA's serial chain of rows -- the pass's critical path -- has the schedulers to
// itself.  The CTA never waits for a systolic warp, so this cannot deadlock; it ends when the CTA has no ticket left.
static __device__ __noinline__ void wait_row_cta(const unsigned long long *counters)
{
    unsigned smid;
    asm("mov.u32 %0, %%smid;" : "=r"(smid));
    const volatile unsigned long long *busy = counters + CNT_ROW_BUSY + (smid & 255u);
    while (*busy != 0ULL) __nanosleep(20000);
}

template <bool TB, bool COOP>
__global__ void __launch_bounds__(SFE_BLOCK_THREADS, SFE_MIN_BLOCKS) ydrop_kernel(const YdParams p)
{
    extern __shared__ __align__(16) char smem[];
    const int lane = sfe_lane();
    char *wsm = smem + (threadIdx.x >> 5) * SFE_WARP_SMEM;
    // re-run passes after a traceback-arena overflow admit only as many warps as the arena can serve
    if ((int)(blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5)) >= p.max_warps) return;
    if (COOP) {
        // start gate: the row kernel's CTAs were launched on another stream and must be RESIDENT before this kernel's
        // persistent blocks take the SMs (else they start when these blocks leave: the two kernels run one after the other).
        // This launch leaves room for them (2 blocks per SM), so they always arrive; the wait is bounded all the same.
        const volatile unsigned long long *started = &p.counters[CNT_ROW_STARTED];
        for (int spin = 0; spin < 20000 && *started < (unsigned long long)p.row_grid; spin++) __nanosleep(1000);
    }
    // Ticket queue (a3): tickets are sorted longest bin first and every warp takes the next one (LPT order).
    // One extension is a serial chain of wavefront steps (R4 allows only 32 rows in flight), so the longest
    // halves decide when the kernel ends -- and the SM's schedulers strongly favour the lowest hardware warp
    // slots (measured with sfe_last_half_profile: 140 cycles per step in slots 0-3, 310 in slots 16-19, 18 warps
    // resident).  The longest tickets are therefore reserved: segment k (n_sm x 4 tickets) is served first by
    // the warps of slot class k = slot / 4, k = 0..3; then everybody drains the main queue and, at the end,
    // whatever is left in any segment.
    unsigned wslot;
    asm("mov.u32 %0, %%warpid;" : "=r"(wslot));
    const long long seg = p.seg_tickets;
    const int my_class = (int)(wslot >> 2);
    const int ncls = p.n_classes;                      // slot classes of this launch (1..4): segments 0 .. ncls-1 are reserved
    // the first counters[CNT_ROW_N] tickets (the longest) belong to the cooperative row kernel launched beside this one
    const long long base = p.row_split ? (long long)*((volatile unsigned long long *)&p.counters[CNT_ROW_N]) : 0;
    for (int phase = 0; phase < 6; phase++) {
        // phase 0: my class's segment; phase 1: main queue; phases 2..5: leftovers of segments 0..3
        const int k = phase == 0 ? my_class : phase - 2;
        if (phase != 1 && (k >= ncls || seg == 0)) continue;
        const long long lo0 = base + (phase == 1 ? (seg ? ncls * seg : 0) : k * seg);
        const long long lo = lo0 < p.n_tickets ? lo0 : p.n_tickets;
        const long long hi = phase == 1 ? p.n_tickets : (lo + seg < p.n_tickets ? lo + seg : p.n_tickets);
        unsigned long long *cnt = &p.counters[phase == 1 ? CNT_TICKET : CNT_CLASS0 + k];
        for (;;) {
            if (COOP) wait_row_cta(p.counters);
            unsigned long long tk = 0;
            if (lane == 0) tk = atomicAdd(cnt, 1ULL);
            tk = __shfl_sync(FULL, tk, 0);
            if (lo + (long long)tk >= hi) break;
            // the reserved (longest) tickets run with a lane skew of 2: a shorter dependent step, a few more idle steps
            bool done = false;
            const bool long_skew = phase == 0 && SFE_LONG_SKEW == 2;
            if (long_skew) done = extend_half<TB, SFE_RING_LOG2, false, SFE_LONG_SKEW, COOP>(p, p.tickets[lo + tk], wsm, wsm, lane, SFE_ST_SKEW2);
            if (!done) extend_half<TB, SFE_RING_LOG2, false, 1, COOP>(p, p.tickets[lo + tk], wsm, wsm, lane, long_skew ? SFE_ST_SKEW_RETRY : 0u);
            __syncwarp();
        }
    }
}

// Runs in stream order right after the systolic kernel of a hand-off pass: tells the row-kernel CTAs serving the queue on the
// other stream that no more entries will come.  (Counting the leaving warps inside ydrop_kernel itself cost its hot loop
// registers: spills, +20 % on C4.)
__global__ void mark_sys_done_kernel(unsigned long long *counters, unsigned long long n)
{
    __threadfence();
    *((volatile unsigned long long *)&counters[CNT_SYS_DONE]) = n;
}

// Halves whose strip outgrew the shared-memory window (status SFE_ST_WIDE_PENDING) are collected ...
__global__ void select_wide_kernel(const YdParams p)
{
    const long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (x >= p.n_tickets) return;
    const int hid = p.tickets[x];
    if (p.halves[hid].status & SFE_ST_WIDE_PENDING) p.wide_tickets[atomicAdd(&p.counters[CNT_WIDE_N], 1ULL)] = hid;
}

// ... and re-run, bit-exactly the same algorithm, with 2^16-column rings in global memory (one warp per
// block, always launched: the ticket count is read on the device, so no host synchronisation).
template <bool TB>
__global__ void __launch_bounds__(32) ydrop_wide_kernel(const YdParams p)
{
    __shared__ __align__(16) char wk[SFE_WALK_SMEM];         // traceback-walk window + ops staging (the rings are in global memory)
    const int lane = sfe_lane();
    char *wsm = p.wide_ring + (size_t)blockIdx.x * RingGeom<SFE_WIDE_RING_LOG2>::WARP_BYTES;
    const long long n = (long long)*((volatile unsigned long long *)&p.counters[CNT_WIDE_N]);
    for (;;) {
        unsigned long long tk = 0;
        if (lane == 0) tk = atomicAdd(&p.counters[CNT_WIDE_TICKET], 1ULL);
        tk = __shfl_sync(FULL, tk, 0);
        if ((long long)tk >= n) break;
        extend_half<TB, SFE_WIDE_RING_LOG2, true, 1>(p, p.wide_tickets[tk], wsm, wk, lane, 0u);
        __syncwarp();
    }
}

int sfe_launch_long_left(const YdParams &p, bool want_tb, int n_sm, cudaStream_t st);
int sfe_launch_ydrop_block(const YdParams &p, bool want_tb, int n_sm, cudaStream_t st);
int sfe_launch_ydrop_row(const YdParams &p, bool want_tb, long long grid, cudaStream_t st);

// Function attributes are per DEVICE: sfe_create calls this after cudaSetDevice, for every context.
int sfe_ydrop_init_device(void)
{
    const int smem = (SFE_BLOCK_THREADS / 32) * SFE_WARP_SMEM;
    SFE_CUDA_CHECK(cudaFuncSetAttribute(ydrop_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    SFE_CUDA_CHECK(cudaFuncSetAttribute(ydrop_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    SFE_CUDA_CHECK(cudaFuncSetAttribute(ydrop_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    SFE_CUDA_CHECK(cudaFuncSetAttribute(ydrop_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    return SFE_OK;
}

// use_block: the whole pass goes to the row-synchronous block kernel (ydrop_block_kernel.cu) instead of the
// warp-systolic one; either way halves whose band outgrew the window are re-run by the wide kernel.
// use_block: every half on a cooperative kernel (the row kernel; Lambda = 0: the first block kernel).  Otherwise the
// warp-systolic kernel, and -- row_split -- the row kernel beside it on `aux` for the first counters[CNT_ROW_N] (longest)
// tickets; fork / join through the two events.
int sfe_launch_ydrop(const YdParams &p_in, bool want_tb, bool use_block, int n_sm, cudaStream_t st, cudaStream_t aux,
                     cudaEvent_t ev_fork, cudaEvent_t ev_join)
{
    YdParams p = p_in;
    p.n_classes = 4;
    const bool split = !use_block && p.row_split && aux != nullptr;
    if (!split) p.row_split = 0;
    if (use_block) {
        int rc;
        if (p.lag0) rc = sfe_launch_ydrop_block(p, want_tb, n_sm, st);
        else { p.row_all = 1; rc = sfe_launch_ydrop_row(p, want_tb, p.n_tickets < 2LL * n_sm ? p.n_tickets : 2LL * n_sm, st); }
        if (rc) return rc;
    } else {
        int warps_per_block = SFE_BLOCK_THREADS / 32;
        size_t smem = (size_t)warps_per_block * SFE_WARP_SMEM;
        int bps = 0;
        if (want_tb) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, ydrop_kernel<true, false>, SFE_BLOCK_THREADS, smem);
        else cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, ydrop_kernel<false, false>, SFE_BLOCK_THREADS, smem);
        if (bps < 1) return SFE_ECUDA;
        long long blocks;
        if (p.sparse_warps > 0) {
            // A pass whose time is its longest half (sfe_speculate's batches): one extension is a serial chain of wavefront
            // steps and every co-resident warp on its scheduler slows it down (solo step 49 / 77 cycles, 140-310 with 18
            // warps per SM).  Blocks of 4 warps = one warp per SM sub-partition; sparse_warps / 4 blocks per SM.
            warps_per_block = 4;
            smem = (size_t)warps_per_block * SFE_WARP_SMEM;
            int per_sm = (p.sparse_warps + 3) / 4;
            if (per_sm < 1) per_sm = 1;
            if (per_sm > 4) per_sm = 4;
            blocks = (long long)n_sm * per_sm;
            p.n_classes = per_sm;                             // warp slots 0 .. 4 per_sm - 1 exist: that many reserved segments
        } else {
            // A pass with at most one ticket per warp slot ends with its longest half: fewer resident warps make every half
            // faster (measured on the windowed workloads: 12 warps per SM beat 18 by 7-12 %, 6 are too few).
            if (bps > 2 && p.n_tickets <= (long long)n_sm * bps * warps_per_block) bps = 2;
            blocks = (long long)n_sm * bps;
        }
        if ((split || (p.long_strips > 0 && aux != nullptr && p.row_slots > 0)) && p.sparse_warps == 0 && bps > 2) {
            bps = 2;                                              // beside the row kernel: 2 blocks + one row CTA fill an SM's registers
            blocks = (long long)n_sm * bps;
        }
        const long long need = (p.n_tickets + warps_per_block - 1) / warps_per_block;
        if (blocks > need) blocks = need;
        if (blocks < 1) blocks = 1;
        // hand-off of long halves: row-kernel CTAs serve a queue beside this kernel (never all SMs: the systolic blocks must
        // always find room, the serving CTAs wait for them to finish)
        const bool handoff = !split && p.long_strips > 0 && aux != nullptr && p.row_slots > 0 && p.max_warps == 0x7fffffff;
        if (!handoff) p.long_strips = 0;
        if (handoff) {
            if (p.row_slots > n_sm / 2) p.row_slots = n_sm / 2;
            p.sys_warps = (int)(blocks * warps_per_block);
            SFE_CUDA_CHECK(cudaMemsetAsync(p.long_tickets, 0xff, (size_t)p.n_tickets * sizeof(int32_t), st));
        }
        if (split || handoff) {                                   // launched FIRST so that its CTAs get their SM resources
            SFE_CUDA_CHECK(cudaEventRecord(ev_fork, st));
            SFE_CUDA_CHECK(cudaStreamWaitEvent(aux, ev_fork, 0));
            YdParams pr = p;
            pr.row_all = handoff ? 2 : 0;
            const long long grid = handoff ? (long long)p.row_slots : (p.n_tickets < (long long)n_sm ? p.n_tickets : (long long)n_sm);
            p.row_grid = pr.row_grid = (int)grid;
            const int rc = sfe_launch_ydrop_row(pr, want_tb, grid, aux);
            if (rc) return rc;
            SFE_CUDA_CHECK(cudaEventRecord(ev_join, aux));
        }
        if (split || handoff) {                                   // the variant that waits for / hands over to the row kernel's CTAs
            if (want_tb) SFE_KL ydrop_kernel<true, true><<<(unsigned)blocks, warps_per_block * 32, smem, st>>>(p);
            else SFE_KL ydrop_kernel<false, true><<<(unsigned)blocks, warps_per_block * 32, smem, st>>>(p);
        } else {
            if (want_tb) SFE_KL ydrop_kernel<true, false><<<(unsigned)blocks, warps_per_block * 32, smem, st>>>(p);
            else SFE_KL ydrop_kernel<false, false><<<(unsigned)blocks, warps_per_block * 32, smem, st>>>(p);
        }
        if (handoff) SFE_KL mark_sys_done_kernel<<<1, 1, 0, st>>>(p.counters, (unsigned long long)p.sys_warps);
        if (split || handoff) SFE_CUDA_CHECK(cudaStreamWaitEvent(st, ev_join, 0));
        if (handoff) {
            const int rc = sfe_launch_long_left(p, want_tb, n_sm, st);
            if (rc) return rc;
        }
    }
    const int bs = 256;
    SFE_KL select_wide_kernel<<<(unsigned)((p.n_tickets + bs - 1) / bs), bs, 0, st>>>(p);
    if (want_tb) SFE_KL ydrop_wide_kernel<true><<<SFE_WIDE_WARPS, 32, 0, st>>>(p);
    else SFE_KL ydrop_wide_kernel<false><<<SFE_WIDE_WARPS, 32, 0, st>>>(p);
    SFE_LAUNCH_CHECK();
}
