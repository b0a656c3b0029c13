// sfe_internal.cuh -- shared declarations of the CUDA side of libsfe (sm_100a only).
// Nothing here is shared with oracle/: the oracle defines its own structs and rules.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/sfe.h"

#define SFE_NEG (-(1 << 30))            // "minus infinity" of the DP (R6)
#define SFE_T_INF (-(1 << 29))          // threshold used for SFE_YDROP_INF (R27): every real cell is above it
#define SFE_ST_WIDE_PENDING 0x200u    // internal: the strip outgrew the shared-memory window; re-run by the wide kernel
#define SFE_ST_PASS_OVERFLOW 0x100u   // internal: the traceback arena ran out during this pass; the anchor is re-run
#define SFE_ST_OPS_OVERFLOW 0x400u    // internal: the ops arena ran out; reported as SFE_ST_CIGAR_OVERFLOW
#define SFE_ST_BLOCK 0x800u           // internal: computed by the row-synchronous block kernel
#define SFE_ST_SKEW2 0x1000u          // internal (profile only): the half ran with the lane skew of 2 (reserved ticket)
#define SFE_ST_LONG_PENDING 0x4000u  // internal: a systolic half reached long_strips strips and was handed to the row kernel (re-run there)
#define SFE_ST_SKEW_RETRY 0x2000u     // internal (profile only): a skew-2 strip outgrew the window; re-run with skew 1
// R25: scores stay below 2^29 (inactive-row threshold, SFE_T_INF, the out-of-bounds score and SFE_NEG arithmetic all rely on
// it).  The running best is tested once per strip / per row; it can rise by at most 32 rows x 127 between two tests.
#define SFE_SCORE_LIMIT ((1 << 29) - (1 << 22))
#define SFE_OOB_SCORE 0xE0000000u       // substitution "score" of a column beyond the target end (-2^29)

// ---- shared-memory geometry of one warp -------------------------
// A strip is 32 consecutive DP rows, one per lane, swept left to right; lane l is SK (1 or 2) columns
// behind lane l-1.  Messages (H-(O+X) gated by alive, E) travel lane l -> l+1 through a tiny
// exchange area; the last lane's messages go to the boundary ring that lane 0 of the NEXT strip
// reads.  Everything is laid out in 8 "rows"; step k of an unrolled group of 16 steps uses row k & 7
// (and, in the ring, segment base + (k >> 3)), so that every access in the unrolled loop is
// base + immediate.
// The ring capacity is a template parameter: 2^10 columns in shared memory for the normal kernel,
// 2^16 columns in global memory (L2) for the wide-band kernel that re-runs the rare halves whose
// strip exceeds the shared-memory window.
#define SFE_EXCH_BYTES 256                          // 32 lanes x 8 B
#define SFE_RING_LOG2 10
#define SFE_WIDE_RING_LOG2 16
template <int RL2> struct RingGeom {
    static constexpr int RING = 1 << RL2;                        // boundary-ring capacity in columns
    static constexpr int ROW_STRIDE = SFE_EXCH_BYTES + RING;     // bytes: exchange area + RING/8 segments x 8 B
    static constexpr int SELRING = RING;                         // selector ring (>= MAX_STEPS + 192: the next strip re-reads the window start)
    static constexpr int WARP_BYTES = 8 * ROW_STRIDE + (SELRING + 32) * 2;
    static constexpr int MAX_STEPS = RING - 192;                 // a strip wider than this bails out (multiple of 16)
};
#define SFE_WARP_SMEM (RingGeom<SFE_RING_LOG2>::WARP_BYTES)
#define SFE_WIDE_WARPS 148                          // warps of the wide-band kernel (one per block)

// ---- traceback arena --------------------------------------------------------------------------
// Record = 32 lanes x two 32-bit words (16 cells x 4 bits) = 256 B, written coalesced (one 8-byte
// store per lane) by one warp per group of 16 steps; lane l owns words 2l (bit planes 3 and 2 of its
// 16 cells: plane 3 in the upper half, step k at bit 15 - k) and 2l+1 (planes 1 and 0).  Records live in 64 KiB chunks handed out by an atomic counter; a half's chunks
// form a backward-linked list (chunk_prev).
// Chunks are recycled: a lock-free ring of free chunk ids (SfeFreeRing) hands them out and takes them
// back as soon as the warp that filled them has walked its traceback, so the arena only has to hold
// what the resident warps need at the same time.
#define SFE_REC_WORDS 64
#define SFE_REC_BYTES (SFE_REC_WORDS * 4)
#define SFE_CHUNK_RECS 256
#define SFE_CHUNK_BYTES (SFE_CHUNK_RECS * SFE_REC_BYTES)

// ---- CIGAR staging ------------------------------------------------------------------------------
// The warp that computed a half walks its traceback right away (ydrop_kernel.cu, walk_traceback) and
// stages the run-length ops, in walk order (end cell -> origin), as segments in the ops arena:
//   word 0 = offset of the previous segment of the same half (SFE_NO_SEG if none), word 1 = number
//   of ops, then the ops.  emit_kernel copies them to their final, anchor-ordered place (a8).
#define SFE_NO_SEG 0xffffffffu
#define SFE_WALK_WIN_RECS 8                         // traceback records held in shared memory while walking
#define SFE_WALK_OPS 512                            // ops staged in shared memory between flushes
#define SFE_WALK_SMEM (SFE_WALK_WIN_RECS * SFE_REC_BYTES + SFE_WALK_OPS * 4)

struct sfe_half {                 // result of one one-sided extension (a7)
    int32_t score;
    int32_t end_i, end_j;         // argbest, rows / columns relative to the anchor
    uint32_t status;
    unsigned long long cells;     // R28
    uint32_t ops_seg;             // offset of the last staged segment in the ops arena, SFE_NO_SEG if none
    int32_t n_ops;                // run-length ops of this half (valid even if they could not be staged)
    int32_t n_strips;
    int32_t n_rec;                // traceback records written
    int32_t steps;                // warp wavefronts executed
    int32_t max_steps;            // widest strip
    long long cycles;             // SM clock cycles from ticket to result (DP + traceback walk)
    uint32_t smid, wslot;         // SM and hardware warp slot that ran it
};

enum { CNT_TICKET = 0, CNT_RING_DROPS, CNT_OVERFLOW, CNT_TBBYTES, CNT_STEPS, CNT_WIDE, CNT_RERUN, CNT_WIDE_N, CNT_WIDE_TICKET, CNT_OPS, CNT_MAXNEED, CNT_CLASS0, CNT_CLASS1, CNT_CLASS2, CNT_CLASS3, CNT_BLOCK_HALVES,
       CNT_ROW_N, CNT_ROW_TICKET,
       CNT_LONG_N, CNT_LONG_TICKET,  // hand-off queue (long_tickets): entries pushed by the systolic kernel / positions drawn by idle row CTAs
       CNT_ROW_FREE, CNT_SYS_DONE,   // row CTAs idle and not yet claimed (signed) / systolic warps that have left their kernel
       CNT_LONG_LEFT,                // hand-offs nobody served (safety net, normally 0): re-run after the two kernels
       CNT_ROW_STARTED,              // CTAs of the row kernel beside the systolic one that have started (the systolic kernel's start gate)
       CNT_ROW_BUSY = 24,            // + (smid & 255): row-kernel CTAs at work on that SM (the systolic warps there wait: see ydrop_kernel)
       CNT_N = 24 + 256 };

struct SfeFreeRing {              // persistent across launches: every half returns its chunks before it ends
    unsigned long long head;      // pops issued
    unsigned long long tail;      // pushes issued
    long long avail;              // chunks that may still be popped (decremented before head moves)
};

struct YdParams {
    const uint8_t *t_codes, *t_nmask;
    const uint8_t *q_codes, *q_nmask, *qrc_codes, *qrc_nmask;
    long long t_len, q_len;
    const sfe_pair *pairs;
    const sfe_anchor *anchors;
    const int32_t *tickets;       // half ids (2*anchor + dir), in issue order
    long long n_tickets;
    long long seg_tickets;        // tickets reserved per warp-slot class (0 = no reservation), see ydrop_kernel
    unsigned long long *counters; // CNT_*
    sfe_half *halves;             // [2 * n_anchors]
    uint32_t *pool;               // traceback arena
    int32_t *chunk_prev;
    int32_t *free_ring;           // n_chunks slots: a chunk id, or -1 while the slot is empty
    SfeFreeRing *ring_state;
    int32_t n_chunks;
    int32_t max_warps;            // warps of the normal kernel allowed to work in this pass
    int32_t row_all;              // row kernel: 1 = every ticket; 0 = the first counters[CNT_ROW_N] (the longest); 2 = serve the hand-off queue
                                  // while the systolic kernel runs; 3 = long_tickets[n_tickets .. + counters[CNT_LONG_LEFT]) (leftovers)
    int32_t long_strips;          // systolic kernel: > 0 = hand-off check-points at long_strips, 2 long_strips, 4 long_strips ... 32-row strips
    int32_t row_slots;            // CTAs of the row kernel serving the queue (reserve rule of the check-points)
    int32_t sys_warps;            // warps of the systolic kernel of this pass (the serving CTAs leave when all of them have)
    int32_t row_grid;             // CTAs of the row kernel launched beside the systolic kernel (its start gate waits for them)
    int32_t *long_tickets;        // [2 n_tickets]: the hand-off queue (-1 = not written yet), then the leftovers
    int32_t row_split;            // systolic kernel: 1 = skip the first counters[CNT_ROW_N] tickets (the row kernel takes them)
    int32_t n_classes;            // reserved ticket segments in use (set by sfe_launch_ydrop: 4, or fewer in a sparse launch)
    int32_t sparse_warps;         // > 0: resident warps per SM for a chain-bound pass (blocks of 4 warps), see sfe_launch_ydrop
    int32_t n_pairs;
    int32_t OX, X, Y, ydrop_inf;
    int32_t lag0;                 // prune_lag == 0 (R4, serial-order pruning): block kernel only
    uint32_t srow[5];             // packed int8 scores of a query base A,C,G,T,N against A,C,G,T
    uint32_t srow_hi;             // bytes: n_score, 0x00, 0xE0 (OOB), 0x00
    char *wide_ring;              // global-memory rings of the wide-band kernel: SFE_WIDE_WARPS x RingGeom<16>::WARP_BYTES
    int32_t *wide_tickets;        // halves that bailed out of the normal kernel in this pass
    uint32_t *ops_stage;          // ops arena (segments, see above); counters[CNT_OPS] = words used
    unsigned long long ops_cap;   // capacity of the ops arena in words
};

static __device__ __forceinline__ int sfe_lane() { return threadIdx.x & 31; }

// base k of a packed sequence: code 0..3, or 4 if the N-mask bit is set
static __device__ __forceinline__ int sfe_base(const uint8_t *codes2, const uint8_t *nmask, long long k)
{
    const int c = (codes2[k >> 2] >> ((k & 3) * 2)) & 3;
    const int n = (nmask[k >> 3] >> (k & 7)) & 1;
    return n ? 4 : c;
}

// kernel launches enqueued by the calling host thread (read through sfe_launch_counter); SFE_KL prefixes every launch
extern thread_local long long sfe_tls_launches;
#define SFE_KL (++sfe_tls_launches),

// last CUDA failure of the calling host thread (file:line + runtime message), readable through sfe_last_error_detail()
void sfe_note_cuda_error(cudaError_t e, const char *file, int line);
void sfe_note_error_text(const char *msg);                 // the text sfe_last_error_detail returns (calling host thread)
#define SFE_CUDA_CHECK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { sfe_note_cuda_error(e_, __FILE__, __LINE__); return SFE_ECUDA; } } while (0)
#define SFE_LAUNCH_CHECK() do { cudaError_t e_ = cudaGetLastError(); if (e_ != cudaSuccess) { sfe_note_cuda_error(e_, __FILE__, __LINE__); return SFE_ECUDA; } return SFE_OK; } while (0)
