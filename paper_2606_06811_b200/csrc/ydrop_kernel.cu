// ydrop_kernel.cu -- the warp-systolic Y-drop gapped extension.
//
// One warp = one one-sided extension ("anchor-half").  The paper's kernel
// (Fig. 8) gives each thread one line of the DP matrix and passes neighbour values
// between threads; this kernel keeps that systolic idea but is organised for sm_100a:
//   * rows are processed in strips of 32 (lane l owns row 32 s + l), each lane sweeping its row
//     left to right one column behind the lane above, so that 32 lanes stay busy whatever the
//     width of the live band is (the band is 0..~700 columns wide and changes every row);
//   * per cell: PRMT score lookup from a packed int8 row, IADD3, two VIADDMNMX (E, F), one
//     VIMNMX3 (H) -- the Blackwell DPX instructions -- plus compare/select for the Y-drop prune;
//   * lane-to-lane messages and the strip-to-strip boundary row go through a 10 KiB per-warp
//     shared-memory area laid out so that every access of the 8x unrolled loop is base+immediate;
//   * 4 traceback bits per cell are packed 8 cells to a word and written as one coalesced 128 B
//     record per warp per 8 steps into the HBM arena (R11);
//   * rows are pruned with the row-lagged threshold T(r) = best(rows <= r - 32) - ydrop (R4),
//     which is exactly what is final when row r starts in this schedule.
// Dead cells are gated only on the diagonal/open edge (R6 lemma).
#include "sfe_internal.cuh"

#define FULL 0xffffffffu
#define SFE_BLOCK_THREADS 192     // 6 warps x 12.3 KB of shared memory; 3 blocks = 18 warps per SM
#define ST_PASS_OVERFLOW 0x100u   // internal: traceback arena ran out during this pass

// PRMT with the sign-replicate selector mode (bit 3 of a selector nibble), which __byte_perm masks off
static __device__ __forceinline__ int prmt_sx(uint32_t lo, uint32_t hi, uint32_t sel)
{
    int r;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(r) : "r"(lo), "r"(hi), "r"(sel));
    return r;
}

template <int RL2>
static __device__ __forceinline__ int bnd_off(int c)
{
    const int u = c + 7;
    return (u & 7) * RingGeom<RL2>::ROW_STRIDE + SFE_EXCH_BYTES + ((u >> 3) & (RingGeom<RL2>::RING / 8 - 1)) * 8;
}

struct HalfGeom {
    const uint8_t *qc, *qm, *tc, *tm;
    long long q0, t0;     // base index of row i / column j is q0 + d*i, t0 + d*j (i, j >= 1)
    int d;
    int n, m;
};

static __device__ __forceinline__ uint32_t col_selector(const HalfGeom &g, int c)
{
    if (c <= 0) return 0x8880u;
    if (c > g.m) return 0x6555u;                         // -> SFE_OOB_SCORE
    const int b = sfe_base(g.tc, g.tm, g.t0 + (long long)g.d * c);
    return b == 4 ? 0xCCC4u : 0x8880u + 0x1111u * (uint32_t)b;
}

// fill selector-ring entries for columns [lo, hi)
template <int RL2>
static __device__ __forceinline__ void fill_sel(uint16_t *selring, const HalfGeom &g, int lo, int hi, int lane)
{
    for (int c = lo + lane; c < hi; c += 32) {
        const uint16_t v = (uint16_t)col_selector(g, c);
        const int idx = c & (RingGeom<RL2>::SELRING - 1);
        selring[idx] = v;
        if (idx < 8) selring[idx + RingGeom<RL2>::SELRING] = v;
    }
    __syncwarp();
}

// fill boundary-ring entries for columns [lo, hi) with "dead"
template <int RL2>
static __device__ __forceinline__ void fill_bnd_neg(char *wbase, int lo, int hi, int lane)
{
    for (int c = lo + lane; c < hi; c += 32) *(int2 *)(wbase + bnd_off<RL2>(c)) = make_int2(SFE_NEG, SFE_NEG);
    __syncwarp();
}

struct TbWriter {
    uint32_t *pool; int32_t *chunk_prev; unsigned long long *counters; int n_chunks;
    uint32_t *ptr;          // this lane's word of the next record
    int left;               // records left in the current chunk
    int cur_chunk; int nrec; bool ok;
    __device__ __forceinline__ void put(uint32_t word, int lane)
    {
        if (!ok) return;
        if (left == 0) {
            int c = 0;
            if (lane == 0) c = (int)atomicAdd(&counters[CNT_CHUNK], 1ULL);
            c = __shfl_sync(FULL, c, 0);
            if (c >= n_chunks) { ok = false; return; }
            if (lane == 0) chunk_prev[c] = cur_chunk;
            cur_chunk = c;
            ptr = pool + (size_t)c * SFE_CHUNK_RECS * 32 + lane;
            left = SFE_CHUNK_RECS;
        }
        *ptr = word;
        ptr += 32; left--; nrec++;
    }
};

// Integer adds forced onto the FMA pipe (IMAD): the ALU pipe is the binding resource of this kernel
// (profiles/r1_01), the FMA pipe is otherwise idle.
static __device__ __forceinline__ int fma_add(int a, int b)
{
    int r;
    asm("mad.lo.s32 %0, %1, 1, %2;" : "=r"(r) : "r"(a), "r"(b));
    return r;
}
// (a & ~b) | (c & b) in one LOP3
static __device__ __forceinline__ int lop3_sel(int a, int b, int c)
{
    int r;
    asm("lop3.b32 %0, %1, %2, %3, 0xB8;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
    return r;
}
static __device__ __forceinline__ int fma_mad(int a, int b, int c)   // a * b + c
{
    int r;
    asm("mad.lo.s32 %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
    return r;
}
static __device__ __forceinline__ int fma_sub(int a, int b)      // a - b
{
    int r;
    asm("mad.lo.s32 %0, %1, -1, %2;" : "=r"(r) : "r"(b), "r"(a));
    return r;
}
// acc = (acc << 1) | (sign bit of x): one SHF.L.W
static __device__ __forceinline__ uint32_t shift_in_sign(uint32_t acc, int x) { return __funnelshift_l((uint32_t)x, acc, 1); }

// One group of 8 wavefront steps.  Everything indexed by k is an immediate after unrolling.
// Per cell the ALU pipe sees: PRMT, IADD3 (M), 2 x VIADDMNMX (E, F), VIMNMX3 (H), SHF + LOP3 (alive gate),
// 4 x SHF (traceback bits), SHF + VIMNMX (best); the FMA pipe sees the 8 subtractions / shift-adds.
// Traceback nibble of step k sits at bits 4(7-k)..4(7-k)+3 of acc:
//   bit3 = H not from M, bit2 = H not from E, bit1 = E extended, bit0 = F extended (R11).
// gneg = -(dead-bit pattern): gneg' = 2 gneg + g with g = 0 (alive) / -1 (dead); step k at bit 7-k of -gneg.
// bm shifts in one bit per step: 1 iff that step raised the lane-local best (strict '>', R7).
template <bool TB, bool EDGE, int RL2, bool GLOBAL>
static __device__ __forceinline__ void run_group8(int &upH, int &upE, int &dg, int &F, int &Hgl, int &best, uint32_t &bm,
                                                  uint32_t &acc, int &gneg, const uint32_t srow_lo,
                                                  const uint32_t srow_hi, const int T, const int OX, const int tox,
                                                  const int X, const char *rptr, char *wptr, const uint16_t *selp,
                                                  const int col0, const int m)
{
#pragma unroll
    for (int k = 0; k < 8; k++) {
        const uint32_t sel = GLOBAL ? __ldcg(selp + k) : selp[k];
        const int s = prmt_sx(srow_lo, srow_hi, sel);
        const int M = dg + s + OX;                         // dg = H(i-1,j-1) - OX, or NEG if dead
        const int E = __viaddmax_s32(upE, -X, upH);        // upH = H(i-1,j) - OX, or NEG if dead
        const int Fn = __viaddmax_s32(F, -X, Hgl);         // Hgl = H(i,j-1) - OX (ungated: R6 lemma)
        int H = __vimax3_s32(M, E, Fn);
        if (EDGE) { if (col0 + k > m) H = SFE_NEG; }       // beyond the target end
        const int d = fma_sub(H, T);                       // alive <=> d >= 0 (R5)
        const int Hg = fma_add(d, tox);                    // H - OX, as d + (T - OX) so that it stays an IMAD
        const int gmask = d >> 31;                         // 0 alive, -1 dead
        if (TB) {
            acc = shift_in_sign(acc, fma_sub(M, H));       // M < H  <=> H not from M
            acc = shift_in_sign(acc, fma_sub(E, H));       // E < H  <=> H not from E
            acc = shift_in_sign(acc, fma_sub(upH, E));     // upH < E <=> E extended (open wins ties)
            acc = shift_in_sign(acc, fma_sub(Hgl, Fn));    // Hgl < F <=> F extended
        }
        gneg = fma_mad(gneg, 2, gmask);
        bm = shift_in_sign(bm, fma_sub(best, H));          // best < H <=> new lane-local best
        best = max(best, H);
        const int msgH = lop3_sel(Hg, gmask, SFE_NEG);     // one LOP3: dead cells send NEG
        *(int2 *)(wptr + k * RingGeom<RL2>::ROW_STRIDE) = make_int2(msgH, E);
        dg = upH; F = Fn; Hgl = Hg;
        __syncwarp();
        const int2 u = GLOBAL ? __ldcg((const int2 *)(rptr + k * RingGeom<RL2>::ROW_STRIDE))
                              : *(const int2 *)(rptr + k * RingGeom<RL2>::ROW_STRIDE);
        upH = u.x; upE = u.y;
    }
}

template <bool TB, int RL2, bool GLOBAL>
static __device__ void extend_half(const YdParams &p, const int hid, char *wsm, const int lane)
{
    typedef RingGeom<RL2> G;
    uint16_t *selring = (uint16_t *)(wsm + 8 * G::ROW_STRIDE);
    sfe_half out;
    out.score = 0; out.end_i = 0; out.end_j = 0; out.status = 0; out.cells = 0;
    out.last_hdr = -1; out.last_chunk = -1; out.n_strips = 0; out.n_rec = 0; out.steps = 0; out.max_steps = 0;

    const long long a = hid >> 1;
    const int dir = hid & 1;
    const sfe_anchor an = p.anchors[a];
    HalfGeom g;
    bool bad = an.pair < 0 || an.pair >= p.n_pairs;
    sfe_pair pr = {0, 0, 0, 0};
    if (!bad) pr = p.pairs[an.pair];
    long long qb, qe;
    if (an.strand >= 0) { g.qc = p.q_codes; g.qm = p.q_nmask; qb = pr.q_begin; qe = pr.q_end; }
    else { g.qc = p.qrc_codes; g.qm = p.qrc_nmask; qb = p.q_len - pr.q_end; qe = p.q_len - pr.q_begin; }
    g.tc = p.t_codes; g.tm = p.t_nmask;
    bad = bad || an.tpos < pr.t_begin || an.tpos > pr.t_end || an.qpos < qb || an.qpos > qe || g.qc == nullptr ||
          pr.t_begin < 0 || pr.t_end > p.t_len || qb < 0 || qe > p.q_len;
    if (bad) {
        out.status = SFE_ST_BAD_ANCHOR;
        if (lane == 0) p.halves[hid] = out;
        return;
    }
    long long nn, mm;
    if (dir == 0) { nn = qe - an.qpos; mm = pr.t_end - an.tpos; g.q0 = an.qpos - 1; g.t0 = an.tpos - 1; g.d = 1; }
    else { nn = an.qpos - qb; mm = an.tpos - pr.t_begin; g.q0 = an.qpos; g.t0 = an.tpos; g.d = -1; }
    const long long LIM = 0x7ffffff0LL - 4096;
    g.n = (int)(nn < LIM ? nn : LIM); g.m = (int)(mm < LIM ? mm : LIM);

    const int OX = p.OX, X = p.X;
    TbWriter tb;
    tb.pool = p.pool; tb.chunk_prev = p.chunk_prev; tb.counters = p.counters; tb.n_chunks = p.n_chunks;
    tb.cur_chunk = -1; tb.nrec = 0; tb.ok = TB; tb.ptr = nullptr; tb.left = 0;

    int best = 0, best_i = 0, best_j = 0;     // lane-local first maximum
    int cumA = 0, cumB = 0;                    // lane-local best through the previous strip / the one before
    unsigned long long cells = 0;
    int cs = 0, prevR = -1;
    int bnd_valid = 0;                         // boundary ring holds row (r0-1) for columns < bnd_valid
    int sel_hi = -32;                          // selector ring is filled for columns < sel_hi
    int total_steps = 0, max_steps = 0, last_hdr = -1, n_strips = 0;
    bool wide = false;

    for (int s = 0;; s++) {
        const int r0 = s * 32;
        if (r0 > g.n) break;
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
        const int tox = T - OX;

        if (TB) {   // strip header record: word0 = cs, word1 = previous header's record index
            const int hdr = tb.nrec;
            tb.put(lane == 0 ? (uint32_t)cs : (lane == 1 ? (uint32_t)last_hdr : (uint32_t)s), lane);
            last_hdr = hdr;
        }
        n_strips++;

        if (sel_hi < cs - 32) sel_hi = cs - 32;
        if (bnd_valid <= cs) { fill_bnd_neg<RL2>(wsm, bnd_valid, cs + 64, lane); bnd_valid = cs + 64; }
        int upH = SFE_NEG, upE = SFE_NEG, dg = SFE_NEG, F = SFE_NEG, Hgl = SFE_NEG;
        if (lane == 0) {
            const int2 u = GLOBAL ? __ldcg((const int2 *)(wsm + bnd_off<RL2>(cs))) : *(const int2 *)(wsm + bnd_off<RL2>(cs));
            upH = u.x; upE = u.y;
            if (s == 0) dg = -OX;                           // R8: H(0,0) = 0 enters as the diagonal of (0,0)
        }
        int first_t = 0x7fffffff, last_t = -1, best_t = -1;   // step indices of the first / last alive cell of my row
        uint32_t bm = 0;
        const int best_before = best;
        int t0 = 0;
        bool bail = false;
        const bool is0 = lane == 0, is31 = lane == 31;
        char *const exch_w = wsm + lane * 8;
        const char *const exch_r = wsm + (lane - 1) * 8;
        char *const bnd = wsm + SFE_EXCH_BYTES;
        int gneg = 0;
        for (;; t0 += 8) {
            const int cmax = cs + t0 + 7;                   // lane 0's last column of this group
            if (sel_hi <= cmax) { fill_sel<RL2>(selring, g, sel_hi, cmax + 129, lane); sel_hi = cmax + 129; }
            if (bnd_valid <= cmax + 1) { fill_bnd_neg<RL2>(wsm, bnd_valid, bnd_valid + 64, lane); bnd_valid += 64; }
            const int base8 = (cs + t0) >> 3;
            const char *rptr = is0 ? bnd + ((base8 + 1) & (G::RING / 8 - 1)) * 8 : exch_r;
            char *wptr = is31 ? bnd + ((base8 - 3) & (G::RING / 8 - 1)) * 8 : exch_w;
            const int col0 = cs + t0 - lane;
            const uint16_t *selp = selring + (col0 & (G::SELRING - 1));
            uint32_t acc = 0;
            if (cmax > g.m)
                run_group8<TB, true, RL2, GLOBAL>(upH, upE, dg, F, Hgl, best, bm, acc, gneg, srow_lo, srow_hi, T, OX, tox, X, rptr, wptr,
                                     selp, col0, g.m);
            else
                run_group8<TB, false, RL2, GLOBAL>(upH, upE, dg, F, Hgl, best, bm, acc, gneg, srow_lo, srow_hi, T, OX, tox, X, rptr, wptr,
                                      selp, col0, g.m);
            if (TB) tb.put(acc, lane);
            const uint32_t al = ~(uint32_t)(-gneg) & 0xffu; // alive bits of this group, step k at bit 7-k
            if (bm & 0xffu) best_t = t0 + 8 - __ffs(bm & 0xffu);   // the latest strict increase of this group
            if (al) {
                first_t = min(first_t, t0 + __clz(al) - 24);
                last_t = t0 + 8 - __ffs(al);
            }
            if (!__any_sync(FULL, al != 0) && cs + t0 + 8 > prevR + 1) { t0 += 8; break; }
            if (t0 + 8 >= G::MAX_STEPS) { t0 += 8; bail = true; break; }
        }
        const int first = last_t < 0 ? 0x7fffffff : cs - lane + first_t, last = last_t < 0 ? -1 : cs - lane + last_t;
        total_steps += t0;
        if (t0 > max_steps) max_steps = t0;
        if (bail) { wide = true; break; }
        if (last >= 0) cells += (unsigned long long)(last - first + 1);
        if (best > best_before) { best_i = r; best_j = cs + best_t - lane; }
        cumB = cumA; cumA = best;
        const int L31 = __shfl_sync(FULL, first, 31), R31 = __shfl_sync(FULL, last, 31);
        if (R31 < 0) break;                                 // last row of the strip has no alive cell
        bnd_valid = cs + t0 - 31;                           // lane 31 wrote columns cs-31 .. cs+t0-32
        prevR = R31;
        cs = L31 & ~7;
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

    out.score = bs; out.end_i = bi; out.end_j = bj; out.cells = cells;
    // normal kernel: a bail-out is re-run by the wide kernel; wide kernel: a bail-out is final (band limit)
    out.status = (wide ? (GLOBAL ? (SFE_ST_WIDE | SFE_ST_BAND_LIMIT) : SFE_ST_WIDE_PENDING) : (GLOBAL ? SFE_ST_WIDE : 0u)) |
                 ((TB && !tb.ok) ? ST_PASS_OVERFLOW : 0u);
    out.last_hdr = last_hdr; out.last_chunk = tb.cur_chunk; out.n_strips = n_strips; out.n_rec = tb.nrec;
    out.steps = total_steps; out.max_steps = max_steps;
    if (lane == 0) {
        p.halves[hid] = out;
        atomicAdd(&p.counters[CNT_STEPS], (unsigned long long)total_steps);
        if (TB) atomicAdd(&p.counters[CNT_TBBYTES], (unsigned long long)tb.nrec * 128ULL);
        if (TB && !tb.ok) atomicAdd(&p.counters[CNT_OVERFLOW], 1ULL);
        if (wide && !GLOBAL) atomicAdd(&p.counters[CNT_WIDE], 1ULL);
    }
}

// Persistent kernel: every warp pulls anchor-half tickets from one atomic counter (a3).
template <bool TB>
__global__ void __launch_bounds__(SFE_BLOCK_THREADS) ydrop_kernel(const YdParams p)
{
    extern __shared__ __align__(16) char smem[];
    const int lane = sfe_lane();
    char *wsm = smem + (threadIdx.x >> 5) * SFE_WARP_SMEM;
    for (;;) {
        unsigned long long tk = 0;
        if (lane == 0) tk = atomicAdd(&p.counters[CNT_TICKET], 1ULL);
        tk = __shfl_sync(FULL, tk, 0);
        if ((long long)tk >= p.n_tickets) break;
        extend_half<TB, SFE_RING_LOG2, false>(p, p.tickets[tk], wsm, lane);
        __syncwarp();
    }
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
    const int lane = sfe_lane();
    char *wsm = p.wide_ring + (size_t)blockIdx.x * RingGeom<SFE_WIDE_RING_LOG2>::WARP_BYTES;
    const long long n = (long long)*((volatile unsigned long long *)&p.counters[CNT_WIDE_N]);
    for (;;) {
        unsigned long long tk = 0;
        if (lane == 0) tk = atomicAdd(&p.counters[CNT_WIDE_TICKET], 1ULL);
        tk = __shfl_sync(FULL, tk, 0);
        if ((long long)tk >= n) break;
        extend_half<TB, SFE_WIDE_RING_LOG2, true>(p, p.wide_tickets[tk], wsm, lane);
        __syncwarp();
    }
}

int sfe_launch_ydrop(const YdParams &p, bool want_tb, int n_sm, cudaStream_t st)
{
    const int warps_per_block = SFE_BLOCK_THREADS / 32;
    const size_t smem = (size_t)warps_per_block * SFE_WARP_SMEM;
    static bool attr_done = false;
    if (!attr_done) {
        if (cudaFuncSetAttribute(ydrop_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return SFE_ECUDA;
        if (cudaFuncSetAttribute(ydrop_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return SFE_ECUDA;
        attr_done = true;
    }
    int bps = 0;
    if (want_tb) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, ydrop_kernel<true>, SFE_BLOCK_THREADS, smem);
    else cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, ydrop_kernel<false>, SFE_BLOCK_THREADS, smem);
    if (bps < 1) return SFE_ECUDA;
    long long blocks = (long long)n_sm * bps;
    const long long need = (p.n_tickets + warps_per_block - 1) / warps_per_block;
    if (blocks > need) blocks = need;
    if (blocks < 1) blocks = 1;
    if (want_tb) ydrop_kernel<true><<<(unsigned)blocks, SFE_BLOCK_THREADS, smem, st>>>(p);
    else ydrop_kernel<false><<<(unsigned)blocks, SFE_BLOCK_THREADS, smem, st>>>(p);
    const int bs = 256;
    select_wide_kernel<<<(unsigned)((p.n_tickets + bs - 1) / bs), bs, 0, st>>>(p);
    if (want_tb) ydrop_wide_kernel<true><<<SFE_WIDE_WARPS, 32, 0, st>>>(p);
    else ydrop_wide_kernel<false><<<SFE_WIDE_WARPS, 32, 0, st>>>(p);
    SFE_LAUNCH_CHECK();
}
