/*
 * sfe.h -- C ABI of libsfe: B200 (sm_100a) speculative Y-drop gapped extension.
 *
 * The hot path of arxiv/paper_2606_06811: the gapped-extension (Y-drop) phase of a LASTZ-style
 * seed-filter-extend pipeline run as speculative batches (Algorithm 3), then
 * resolved so that exactly the alignments of the serial in-order loop (PAPER.md:41-72,
 * Algorithm 1) are kept.  The paper names the operations only; the exact recurrence, threshold
 * and tie-break rules are the readings R1..R29 of SURVEY.md 8(c), restated in DESIGN.md.
 *
 * Conventions
 *  - Every function returns int: SFE_OK (0) or a negative SFE_E* code.  No exceptions, no exit(),
 *    nothing printed.
 *  - Pointers named *_dev are DEVICE pointers owned by the caller; *_host are HOST pointers.
 *    Inputs are read-only and must not alias outputs.  The ctx owns only scratch.
 *  - All device work is enqueued on the ctx's CUDA stream.  sfe_pack and sfe_resolve do not
 *    synchronise; sfe_ydrop_batch synchronises the stream once before returning when
 *    SFE_WANT_CIGAR is set (it must read the traceback-overflow counter), otherwise not.
 *  - Coordinates are 0-based corner positions (between bases), int64.  For strand -1 the query
 *    coordinate refers to the reverse-complemented query (R15).
 *  - There is no CPU fallback anywhere in this library.
 */
#ifndef SFE_H
#define SFE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    SFE_OK = 0,
    SFE_EINVAL = -1,   /* bad argument (NULL, negative size, unsupported prune_lag, ...)        */
    SFE_ENOMEM = -2,   /* device or host allocation failed                                      */
    SFE_ECUDA = -3,    /* a CUDA runtime call or kernel launch failed                           */
    SFE_ELIMIT = -4    /* value outside the supported range (see sfe_scoring)                   */
};

#define SFE_YDROP_INF 0x7fffffff      /* R27: no pruning                                        */
#define SFE_PRUNE_LAG 32              /* R4: the row lag the systolic kernel implements exactly; prune_lag = 0
                                         (best so far in row-major order, the serial reading) is accepted
                                         together with SFE_BLOCK_KERNEL                            */

/* flags of sfe_ydrop_batch */
#define SFE_WANT_CIGAR 1u             /* spill traceback pointers to HBM and emit CIGARs         */
#define SFE_SCORE_ONLY 0u             /* scores, boxes and cell counts only                      */
#define SFE_NO_BINNING 2u             /* tickets in anchor order (default: longest-first bins)   */
#define SFE_BLOCK_KERNEL 4u           /* every half on a cooperative-warps kernel (one CTA per half, rows in order, prefix
                                         maximum for F; same results).  SFE_OPT_ROW_KERNEL_CAP > 0
                                         instead hands only a pass's priority tickets to it, beside the systolic kernel   */
#define SFE_NO_BLOCK_KERNEL 8u        /* warp-systolic kernel only (overrides SFE_BLOCK_KERNEL and the default split)     */
#define SFE_CIGAR_KEPT_ONLY 16u       /* sfe_speculate with SFE_WANT_CIGAR: windows run score-only (the commit rule needs
                                         score and box only); CIGARs are produced for the KEPT anchors in one
                                         traceback batch at the end; other anchors get n_ops = 0, cigar_off = -1 */

#define SFE_SPEC_LEADERS 32u          /* sfe_speculate: speculate on PREDICTED LEADERS instead of "the next K uncovered anchors":
                                         an anchor that follows a close earlier anchor on (nearly) the same diagonal is not
                                         extended unless the in-order commit reaches it uncovered; results per anchor are cached.
                                         Same kept set / results as Algorithm 1 for any prediction; far less shadow work.     */

/* per-anchor status bits (sfe_result.status) */
#define SFE_ST_TB_OVERFLOW 1u         /* traceback arena exhausted even when run alone: no CIGAR */
#define SFE_ST_CIGAR_OVERFLOW 2u      /* cigar pool too small: ops not written (n_ops is valid)   */
#define SFE_ST_WIDE 4u                /* informational: a half took the wide-band (global ring) path */
#define SFE_ST_SCORE_LIMIT 8u         /* R25: a half's running best reached 2^29 - 2^22: the half was STOPPED there (its score,
                                         end and box are those of the truncated extension; no CIGAR).  Split the pair.  */
#define SFE_ST_BAD_ANCHOR 16u         /* anchor outside its pair's limits: nothing computed          */
#define SFE_ST_BAND_LIMIT 32u         /* live band wider than 65,344 columns: half not computed      */
#define SFE_ST_INTERNAL 64u           /* traceback walk did not reach the origin (a library bug)     */
#define SFE_ST_SKIPPED 128u           /* sfe_speculate: covered before its window, never extended    */

/* CIGAR op word: (length << 4) | code ; M = aligned pair, I = query base vs gap, D = target base
 * vs gap (R12). */
#define SFE_OP_M 0u
#define SFE_OP_I 1u
#define SFE_OP_D 2u

typedef struct sfe_ctx sfe_ctx;       /* opaque: stream, scratch arenas, queue counters          */

/* Scoring (R1, R2, R5, R13, R16).  Supported range: every sub[][] entry and n_score in
 * [-128, 127] (the kernel keeps a query row's scores as packed int8), gap_open >= 0,
 * gap_extend >= 1, gap_open + gap_extend <= 65535, 0 <= ydrop < 2^28 or SFE_YDROP_INF,
 * prune_lag == SFE_PRUNE_LAG, or 0 with SFE_BLOCK_KERNEL; anything else is SFE_ELIMIT / SFE_EINVAL. */
typedef struct {
    int32_t sub[4][4];                /* [query base][target base], A,C,G,T                      */
    int32_t n_score;                  /* any pair involving N                                    */
    int32_t gap_open, gap_extend;     /* a gap of length k costs gap_open + k * gap_extend       */
    int32_t ydrop;
    int32_t prune_lag;                /* Lambda of R4                                            */
    int32_t min_score;                /* tau; used by sfe_resolve             */
} sfe_scoring;

typedef struct { int64_t tpos, qpos; int32_t pair; int32_t strand; /* +1 / -1 */ } sfe_anchor;

/* extension limits: [t_begin, t_end) x [q_begin, q_end) in the FORWARD query frame; for a
 * strand -1 anchor the query interval is mirrored into the reverse-complement frame. */
typedef struct { int64_t t_begin, t_end, q_begin, q_end; } sfe_pair;

typedef struct {
    int32_t score, score_fwd, score_bwd;
    uint32_t status;
    int64_t tstart, tend, qstart, qend;   /* bounding box, corner coordinates, strand frame      */
    int64_t cigar_off;                    /* index of the first op in the cigar pool, -1 if none  */
    int32_t n_ops, n_ops_back;            /* ops = backward half (n_ops_back), then forward half  */
    uint64_t cells;                       /* R28: cells inside the live column bounds, both halves */
} sfe_result;

typedef struct { int64_t tstart, tend, qstart, qend; int32_t strand; int32_t reserved; } sfe_box;

/* counters accumulated by sfe_resolve / sfe_speculate (R29); never reset by the library.
 * waste (shadow work): by count  1 - (n_kept + n_below) / n_extended,
 *                                    by cells  cells_covered / cells_total. */
typedef struct sfe_stats {
    int64_t n_anchors, n_kept, n_covered, n_below;
    uint64_t cells_total, cells_covered;  /* cells of all extended anchors / of covered ones (shadow work) */
    int64_t n_extended;                   /* anchors that went through sfe_ydrop_batch                     */
    int64_t n_windows;                    /* resolve calls / speculative windows                           */
} sfe_stats;

/* Create a context on `device` that enqueues on `cuda_stream` (a cudaStream_t, may be NULL for
 * the default stream).  scratch_bytes sizes the traceback arena (HBM); 0 selects 1 GiB. */
int sfe_create(sfe_ctx **ctx, int device, void *cuda_stream, size_t scratch_bytes);
int sfe_destroy(sfe_ctx *ctx);
const char *sfe_strerror(int code);
/* file:line and CUDA runtime message of the most recent SFE_ECUDA seen by the CALLING HOST THREAD (for diagnosis) */
const char *sfe_last_error_detail(void);
/* cumulative number of CUDA kernel launches this library has enqueued from the calling host thread (every launch
 * site counts itself); bench.py reports the difference over its timed region as gpu_launches. */
int64_t sfe_launch_counter(void);

/* a1 Pack (R13, R14): ASCII (device) -> 2-bit code plane (base k in byte k/4, bits 2(k%4)..; A0 C1
 * G2 T3, N stored as 0) and 1-bit N-mask plane (base k in byte k/8, bit k%8).  If rc_codes2_dev
 * is non-NULL also the reverse-complement planes (3 - code, reversed order).  Output buffers
 * hold (len+3)/4 and (len+7)/8 bytes, rounded up to a multiple of 16 bytes. */
int sfe_pack(sfe_ctx *ctx, const char *ascii_dev, int64_t len, uint8_t *codes2_dev, uint8_t *nmask_dev,
             uint8_t *rc_codes2_dev, uint8_t *rc_nmask_dev);

/* a2-a8 Speculative batch of two-sided Y-drop extensions (Alg. 3 phase 2;
 * one-sided rules: SURVEY 8(c), R1..R12).  For each anchor: one forward and one backward
 * affine-gap extension on one warp each, joined at the anchor.  results_dev[n_anchors] is
 * always written.  With SFE_WANT_CIGAR the ops of anchor i are written to
 * cigar_pool_dev[cigar_off .. cigar_off + n_ops) (anchor order, deterministic offsets) and
 * *cigar_pool_used_dev receives the total; anchors whose ops do not fit get
 * SFE_ST_CIGAR_OVERFLOW.  qrc_* may be NULL if no anchor has strand -1. */
int sfe_ydrop_batch(sfe_ctx *ctx, const uint8_t *t_codes2_dev, const uint8_t *t_nmask_dev, int64_t t_len,
                    const uint8_t *q_codes2_dev, const uint8_t *q_nmask_dev,
                    const uint8_t *qrc_codes2_dev, const uint8_t *qrc_nmask_dev, int64_t q_len,
                    const sfe_pair *pairs_dev, int32_t n_pairs,
                    const sfe_anchor *anchors_dev, int64_t n_anchors,
                    const sfe_scoring *scoring_host, uint32_t flags,
                    sfe_result *results_dev,
                    uint32_t *cigar_pool_dev, int64_t cigar_pool_cap, int64_t *cigar_pool_used_dev);

/* a9 Resolve (Alg. 3 phase 3; R17, R18, R26): in anchor order,
 *   covered(i) = exists accepted box of the same strand containing (tpos_i, qpos_i),
 *   kept(i)    = !covered(i) && score_i >= min_score  -> its box is appended to accepted.
 * keep_dev[i] = 0 covered, 1 kept, 2 below min_score.  accepted_dev / *n_accepted_dev carry the
 * boxes kept in earlier windows in and the extended list out.  With results_dev == NULL this
 * is the phase-1 "is masked" filter: keep_dev[i] = 0 covered, 1 not covered,
 * nothing appended.  stats_dev (may be NULL) is accumulated, not reset.
 * Deviation from SURVEY 8(b), which sketches `sfe_result *accepted_dev`: the accepted set is an array of sfe_box
 * (40 B: the box and its strand).  The rule reads nothing else of a kept result, the strand is not a field of
 * sfe_result, and a driver that carries the set between windows / calls moves 40 B per kept alignment, not 72. */
int sfe_resolve(sfe_ctx *ctx, const sfe_anchor *anchors_dev, const sfe_result *results_dev, int64_t n,
                int32_t min_score, sfe_box *accepted_dev, int64_t accepted_cap, int64_t *n_accepted_dev,
                uint8_t *keep_dev, sfe_stats *stats_dev);

/* sfe_resolve without a context and without any allocation (Alg. 3 phase 3; same rule, same kernels,
 * same outputs as sfe_resolve, byte for byte) -- for callers that cannot call cudaMalloc: code under CUDA graph capture,
 * tight serving loops, harnesses that forbid it.  sfe_create allocates, so this entry point takes the device ordinal and
 * the stream (NULL = default stream) instead of an sfe_ctx; it calls no cudaMalloc / cudaFree / allocating routine.
 * Its scratch (block minima of tpos, the active-box list) is a file-scope __device__ array inside libsfe.so:
 * 2.75 MiB that every GPU which loads the library holds until the process exits.
 * Limits: n <= SFE_STATIC_MAX_ANCHORS and accepted_cap <= SFE_STATIC_MAX_ACCEPTED, else SFE_ELIMIT (nothing launched,
 * sfe_last_error_detail says which); larger inputs go through sfe_resolve, or through consecutive calls on slices
 * of the anchors that carry accepted_dev / n_accepted_dev (R26).  Arguments, layouts, ownership and the meaning of
 * results_dev == NULL are sfe_resolve's; all pointers are device pointers on `device`.  Asynchronous on the stream.
 * Every call on a device shares the one scratch array.  No part of it needs to start at zero (each call overwrites
 * what it reads), so a previous call's leftovers are harmless; but calls that OVERLAP on the GPU -- different streams,
 * host threads or concurrently replayed graphs -- race on it and must be serialised by the caller.
 * sfe_resolve_static_limits reports the two limits and the array's size in bytes (any pointer may be NULL). */
#define SFE_STATIC_MAX_ANCHORS  (1 << 20)
#define SFE_STATIC_MAX_ACCEPTED (1 << 16)
int sfe_resolve_static(int device, void *cuda_stream, const sfe_anchor *anchors_dev, const sfe_result *results_dev,
                       int64_t n, int32_t min_score, sfe_box *accepted_dev, int64_t accepted_cap,
                       int64_t *n_accepted_dev, uint8_t *keep_dev, sfe_stats *stats_dev);
int sfe_resolve_static_limits(int64_t *max_anchors, int64_t *max_accepted, int64_t *scratch_bytes);

/* Algorithm 3 end to end on device buffers.  Repeats until every anchor is decided:
 *   phase 1  scan forward from the cursor: anchors covered by an accepted box are final (keep 0, result
 *            zeroed with SFE_ST_SKIPPED, never extended); the next window_k uncovered anchors form the window;
 *   phase 2  sfe_ydrop_batch on the window (flags as there);
 *   phase 3  the resolve rule in window order; kept boxes are appended to accepted_dev.
 * Anchors must be in anchor order (the order Algorithm 1 would visit them).  The kept set equals
 * Algorithm 1's for every window_k >= 1 (R20, P7); window_k trades waste for parallelism.
 * results_dev / keep_dev have n_anchors entries in anchor order; CIGARs of all extended anchors go to the
 * pool (offsets grow window by window).  accepted_dev / n_accepted_dev as in sfe_resolve (boxes carried in
 * are honoured).  Synchronises the stream once per window (it reads the window size).
 * With SFE_SPEC_LEADERS phase 1 picks predicted leaders (window_k = most extensions per batch; see the flag and
 * sfe_set_option); anchors must then be sorted by target position within a pair for the prediction to be useful
 * (any order is still exact). */
int sfe_speculate(sfe_ctx *ctx, const uint8_t *t_codes2_dev, const uint8_t *t_nmask_dev, int64_t t_len,
                  const uint8_t *q_codes2_dev, const uint8_t *q_nmask_dev,
                  const uint8_t *qrc_codes2_dev, const uint8_t *qrc_nmask_dev, int64_t q_len,
                  const sfe_pair *pairs_dev, int32_t n_pairs,
                  const sfe_anchor *anchors_dev, int64_t n_anchors,
                  const sfe_scoring *scoring_host, uint32_t flags, int64_t window_k,
                  sfe_result *results_dev, uint8_t *keep_dev,
                  uint32_t *cigar_pool_dev, int64_t cigar_pool_cap, int64_t *cigar_pool_used_dev,
                  sfe_box *accepted_dev, int64_t accepted_cap, int64_t *n_accepted_dev, sfe_stats *stats_dev);

/* Tunables of sfe_speculate with SFE_SPEC_LEADERS (defaults in brackets) and of chain-bound launches.  They change how much
 * is extended and how it is scheduled, never a result.  sfe_set_option returns SFE_EINVAL for an unknown key / bad value. */
enum {
    SFE_OPT_LEADER_DIAG_TOL = 0,   /* [48]    follower: |diagonal - predecessor's diagonal| <= tol ...                              */
    SFE_OPT_LEADER_GAP,            /* [2000]  ... and target distance to that predecessor <= gap ...                                */
    SFE_OPT_LEADER_LOOKBACK,       /* [64]    ... among the previous `lookback` anchors (same strand, same pair) ...                */
    SFE_OPT_LEADER_NBREAK,         /* [64]    ... with fewer than nbreak N between them in the target                               */
    SFE_OPT_SPEC_SPAN,             /* [2^20]  look-ahead, in anchors beyond the commit cursor, in which leaders are extended        */
    SFE_OPT_SPEC_ESC_MAX,          /* [64]    cap of the doubling number of anchors force-extended after repeated commit stops;
                                              1 = exactly one anchor per stop, no cold-diagonal sweep either                        */
    SFE_OPT_SPARSE_WARPS,          /* [0]     resident warps per SM for sfe_speculate's leader batches (0 = the dense launch)       */
    SFE_OPT_FORCE_CLASS,           /* [0]     testing: 1 = nobody leads, 2 = everybody leads, 3 = second half of the anchors never  */
    SFE_OPT_PROMOTE_REACH,         /* [65536] after a batch, followers within this target distance of an extended anchor that will  
                                              not cover them (it scored below tau, or they lie beyond its box) become leaders       */
    SFE_OPT_ROW_KERNEL_CAP,        /* [#SMs]  most priority tickets (leaders predicted long, known long extensions: the longest first) a pass
                                              hands to the cooperative row kernel, one CTA per half, beside the systolic kernel; the CTA
                                              claims its SM while it works.  0 = never.  Plain sfe_ydrop_batch has no priorities         */
    SFE_OPT_ROW_KERNEL_SCORE_ONLY, /* [1]     1 = also in score-only passes                                                              */
    SFE_OPT_LONG_ROWS,             /* [0]     hand-off (off by default): in sfe_speculate's batches a half of the systolic kernel still alive
                                              after this many rows (and after 2, 4, 8 times as many) stops if a CTA of the row kernel is
                                              idle (early check-points leave a reserve) and is re-run by that CTA from its start.  For
                                              passes whose priorities are missing or wrong; not combined with the priority split (it
                                              applies to passes without priorities, or with ROW_KERNEL_CAP = 0).  Rounded up to 32 times
                                              a power of two.  Measured: DESIGN.md section 6                                              */
    SFE_OPT_LONG_ROWS_DENSE,       /* [0]     the same for sfe_ydrop_batch's dense launch; 0 = off                                   */
    SFE_OPT_ROW_SLOTS,             /* [64]    CTAs of the row kernel that serve those hand-offs (at most half of the SMs)            */
    SFE_OPT_N
};
int sfe_set_option(sfe_ctx *ctx, int key, int64_t value);
/* counters of the most recent sfe_speculate with SFE_SPEC_LEADERS: [0] extension batches, [1] commit stops (the commit
 * reached an anchor that was neither covered nor extended), [2] anchors force-extended after stops, [3] stops on a
 * cold diagonal (its extended predecessor scored below tau: every anchor of that diagonal ahead is taken at once),
 * [4] followers promoted to leaders after a batch showed that the anchor they follow will not cover them, [5..7] reserved. */
int sfe_last_speculate_info(sfe_ctx *ctx, int64_t info[8]);

/* End-to-end convenience with HOST buffers (bench.py's e2e leg): copies the ASCII sequences and
 * anchors to the device, packs, extends (flags as above), resolves in one window, copies
 * results / keep / ops / stats back and synchronises.  cigar_host may be NULL. */
int sfe_extend_host(sfe_ctx *ctx, const char *t_ascii_host, int64_t t_len, const char *q_ascii_host, int64_t q_len,
                    const sfe_pair *pairs_host, int32_t n_pairs, const sfe_anchor *anchors_host, int64_t n_anchors,
                    const sfe_scoring *scoring_host, uint32_t flags,
                    sfe_result *results_host, uint8_t *keep_host,
                    uint32_t *cigar_host, int64_t cigar_cap, int64_t *cigar_used_host, sfe_stats *stats_host);

/* The same with Algorithm 3's windows (sfe_speculate, window_k >= 1) between the copies. */
int sfe_speculate_host(sfe_ctx *ctx, const char *t_ascii_host, int64_t t_len, const char *q_ascii_host, int64_t q_len,
                       const sfe_pair *pairs_host, int32_t n_pairs, const sfe_anchor *anchors_host, int64_t n_anchors,
                       const sfe_scoring *scoring_host, uint32_t flags, int64_t window_k,
                       sfe_result *results_host, uint8_t *keep_host,
                       uint32_t *cigar_host, int64_t cigar_cap, int64_t *cigar_used_host, sfe_stats *stats_host);

/* Measurement helpers.  sfe_probe_int_issue runs a register-only microbenchmark
 * of the Y-drop kernel's own integer opcode mix on every SM and reports sustained
 * lane-instructions per clock per SM (the R of the integer-issue roofline).  mix: 0 = the
 * kernel's mix (ALU + DPX + IMAD), 1 = ALU-pipe only (SHF/LOP3), 2 = DPX only
 * (VIADDMNMX/VIMNMX3), 3 = IMAD only.  sfe_last_batch_info returns counters of the most recent
 * sfe_ydrop_batch on this ctx: [0] kernel launches, [1] halves run, [2] halves re-run after a
 * traceback overflow, [3] traceback bytes written, [4] DP steps (warp wavefronts) executed,
 * [5] halves that took the wide path, [6] device time of the Y-drop kernel launches in microseconds
 * (CUDA events on the ctx stream; synchronises on the last one), [7] halves computed by the block kernel,
 * [8] traceback chunks dropped or pops abandoned by the free-chunk ring's bounded waits (a capacity leak that should never
 * happen: 0 in every test), [9..11] reserved (0). */
#define SFE_INFO_N 12
int sfe_probe_int_issue(sfe_ctx *ctx, int mix, int iters, double *lane_ops_per_clk_per_sm, double *elapsed_ms);

/* Per-half profile of the most recent sfe_ydrop_batch on this ctx (Fig. 5: the
 * spread of per-anchor extension runtimes is what defeats static load balancing).  Entry 2a is the
 * forward half of anchor a, 2a+1 the backward half.  cycles = SM clock cycles from ticket to
 * result (DP + traceback walk), steps = warp wavefronts, smid / wslot = where it ran; status = the half's status
 * bits plus, for the tests' stratified sampling, 0x800 computed by the block kernel, 0x1000 ran with the lane skew
 * of 2 (a reserved, longest-first ticket), 0x2000 a skew-2 attempt outgrew its window and the half was re-run with
 * skew 1.  Copies min(n, 2 * n_anchors) entries to profile_host; synchronises the stream. */
typedef struct {
    int64_t cells, cycles;
    int32_t steps, n_strips, max_steps, n_ops;
    uint32_t smid, wslot, status, reserved;
} sfe_half_profile;
int sfe_last_half_profile(sfe_ctx *ctx, int64_t n, sfe_half_profile *profile_host);
int sfe_last_batch_info(sfe_ctx *ctx, int64_t info[SFE_INFO_N]);

#ifdef __cplusplus
}
#endif
#endif /* SFE_H */
