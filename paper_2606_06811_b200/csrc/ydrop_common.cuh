// ydrop_common.cuh -- device code shared by the two Y-drop kernels (warp-systolic ydrop_kernel.cu and the
// row-synchronous block kernel ydrop_block_kernel.cu): score lookup, half geometry, the free-chunk ring of the
// traceback arena, and the run-length ops writer.  Included by those two files only.
#pragma once
#include "sfe_internal.cuh"

#define FULL 0xffffffffu
#define SFE_SPIN_LIMIT (1 << 22)       // iterations a ring operation waits for its partner (normally a handful)

// PRMT with the sign-replicate selector mode (bit 3 of a selector nibble), which __byte_perm masks off
static __device__ __forceinline__ int prmt_sx(uint32_t lo, uint32_t hi, uint32_t sel)
{
    int r;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(r) : "r"(lo), "r"(hi), "r"(sel));
    return r;
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

// Geometry of one half (hid = 2 * anchor + direction): which planes, where row 1 / column 1 are, how far the
// pair's limits allow the DP to go (R9, R10, R15).  Returns false for an anchor outside its pair.
static __device__ __forceinline__ bool half_setup(const YdParams &p, const int hid, HalfGeom &g)
{
    const long long a = hid >> 1;
    const int dir = hid & 1;
    const sfe_anchor an = p.anchors[a];
    bool bad = an.pair < 0 || an.pair >= p.n_pairs;
    sfe_pair pr = {0, 0, 0, 0};
    if (!bad) pr = p.pairs[an.pair];
    long long qb, qe;
    if (an.strand >= 0) { g.qc = p.q_codes; g.qm = p.q_nmask; qb = pr.q_begin; qe = pr.q_end; }
    else { g.qc = p.qrc_codes; g.qm = p.qrc_nmask; qb = p.q_len - pr.q_end; qe = p.q_len - pr.q_begin; }
    g.tc = p.t_codes; g.tm = p.t_nmask;
    bad = bad || an.tpos < pr.t_begin || an.tpos > pr.t_end || an.qpos < qb || an.qpos > qe || g.qc == nullptr ||
          pr.t_begin < 0 || pr.t_end > p.t_len || qb < 0 || qe > p.q_len;
    if (bad) return false;
    long long nn, mm;
    if (dir == 0) { nn = qe - an.qpos; mm = pr.t_end - an.tpos; g.q0 = an.qpos - 1; g.t0 = an.tpos - 1; g.d = 1; }
    else { nn = an.qpos - qb; mm = an.tpos - pr.t_begin; g.q0 = an.qpos; g.t0 = an.tpos; g.d = -1; }
    const long long LIM = 0x7ffffff0LL - 4096;
    g.n = (int)(nn < LIM ? nn : LIM); g.m = (int)(mm < LIM ? mm : LIM);
    return true;
}

// Free-chunk ring (sfe_internal.cuh).  Called by the whole warp; lane 0 does the memory operations and
// every loop runs on a broadcast value, so control flow stays warp-uniform (a loop inside a
// lane-divergent region makes ptxas clone the whole DP loop with real WARPSYNCs).  Both spins wait
// for one bounded action of another resident warp (the matching push / pop has already reserved the
// slot), never for work.
// Returns the chunk id, -1 if the arena is empty, -2 if the bounded wait for the pusher ran out (counted by the caller).
static __device__ __forceinline__ int chunk_pop(int32_t *ring, SfeFreeRing *st, int n_chunks, int lane)
{
    long long a = 0; unsigned long long h = 0;
    if (lane == 0) {
        a = (long long)atomicAdd((unsigned long long *)&st->avail, ~0ULL);            // avail--
        if (a <= 0) atomicAdd((unsigned long long *)&st->avail, 1ULL);                // nothing left: undo
        else h = atomicAdd(&st->head, 1ULL);
    }
    a = __shfl_sync(FULL, a, 0);
    if (a <= 0) return -1;
    int32_t *slot = ring + (h % (unsigned long long)n_chunks);
    int id = -1;
    for (int spin = 0; spin < SFE_SPIN_LIMIT; spin++) {     // bounded: a hang must be impossible, whatever happened to the pusher
        if (lane == 0) id = atomicExch(slot, -1);           // take the id and empty the slot in ONE step: a delayed pop can never
        id = __shfl_sync(FULL, id, 0);                      // read an id that a later lap's pop also reads
        if (id >= 0) break;
    }
    return id < 0 ? -2 : id;                                // -2: treated like an empty arena (score-only now, re-run later)
}
static __device__ __forceinline__ void chunk_push(int32_t *ring, SfeFreeRing *st, int n_chunks, int id, unsigned long long *drops, int lane)
{
    unsigned long long t = 0;
    if (lane == 0) t = atomicAdd(&st->tail, 1ULL);
    int32_t *slot = ring + (t % (unsigned long long)n_chunks);
    int old = 0;
    for (int spin = 0; spin < SFE_SPIN_LIMIT; spin++) {     // the pop that owns this slot may not have emptied it yet
        if (lane == 0) old = atomicCAS(slot, -1, id);
        old = __shfl_sync(FULL, old, 0);
        if (old == -1) break;
    }
    if (old != -1) { if (lane == 0) atomicAdd(drops, 1ULL); return; }   // give the chunk up (capacity leak, counted) rather than wait for ever
    if (lane == 0) atomicAdd((unsigned long long *)&st->avail, 1ULL);
}

struct OpsWriter {                      // run-length encoder + staging of the ops in walk order
    uint32_t *buf;                      // SFE_WALK_OPS words of shared memory
    uint32_t *stage; unsigned long long *used; unsigned long long cap;
    int nbuf, nops, cur_op, run; uint32_t prev_seg; bool ok;
    __device__ __forceinline__ void flush(int lane)
    {
        if (nbuf == 0) return;
        __syncwarp();
        if (ok) {
            unsigned long long base = 0;
            if (lane == 0) base = atomicAdd(used, (unsigned long long)(nbuf + 2));
            base = __shfl_sync(FULL, base, 0);
            if (base + (unsigned long long)(nbuf + 2) > cap) ok = false;
            else {
                if (lane == 0) { stage[base] = prev_seg; stage[base + 1] = (uint32_t)nbuf; }
                for (int x = lane; x < nbuf; x += 32) stage[base + 2 + x] = buf[x];
                prev_seg = (uint32_t)base;
            }
        }
        nbuf = 0;
        __syncwarp();
    }
    __device__ __forceinline__ void push(int lane)
    {
        if (lane == 0) buf[nbuf] = ((uint32_t)run << 4) | (uint32_t)cur_op;
        nbuf++; nops++;
        if (nbuf == SFE_WALK_OPS) flush(lane);
    }
    __device__ __forceinline__ void emit(int op, int cnt, int lane)
    {
        if (cnt <= 0) return;
        if (op == cur_op) { run += cnt; return; }
        if (cur_op >= 0) push(lane);
        cur_op = op; run = cnt;
    }
};

