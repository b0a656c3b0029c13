// api.cu -- the C ABI of include/sfe.h: argument validation, scratch management, launch order.
// Every step of the path runs in the kernels of this directory; there is no CPU fallback.
#include <new>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include "sfe_internal.cuh"


// launchers defined next to their kernels
int sfe_launch_ydrop(const YdParams &p, bool want_tb, bool use_block, int n_sm, cudaStream_t st, cudaStream_t aux,
                     cudaEvent_t ev_fork, cudaEvent_t ev_join);
int sfe_launch_join(const sfe_anchor *anchors, const sfe_half *halves, long long n, const long long *sel, long long n_sel,
                    int want_cigar, sfe_result *results, cudaStream_t st);
int sfe_launch_scan_emit(const sfe_half *halves, long long n, const long long *sel, long long n_sel, const uint32_t *stage,
                         sfe_result *results, uint32_t *cigar_pool, long long cap, long long *pool_used, cudaStream_t st);
int sfe_launch_pack(const char *ascii, long long len, uint8_t *codes2, uint8_t *nmask, uint8_t *rc_codes2,
                    uint8_t *rc_nmask, cudaStream_t st);
int sfe_launch_resolve(const sfe_anchor *anchors, const sfe_result *results, long long n, int min_score, sfe_box *accepted,
                       long long accepted_cap, long long *n_accepted_io, uint8_t *keep, sfe_stats *stats, long long *blkmin,
                       sfe_box *act, cudaStream_t st);
int sfe_launch_tickets(const sfe_anchor *anchors, long long n_anchors, const sfe_pair *pairs, int n_pairs, long long q_len,
                       bool binned, const uint8_t *prio, unsigned int *hist, int32_t *tickets, unsigned long long *counters,
                       long long cap_prio, long long cap_plain, cudaStream_t st);
int sfe_launch_specl_prepare(const sfe_anchor *anchors, long long n, const uint8_t *t_nmask, long long t_len, const uint8_t *q_nmask,
                             const uint8_t *qrc_nmask, long long q_len, int tol, long long gap, int lookback, int n_break,
                             uint8_t *cls, uint8_t *lead_prio, uint8_t *ext_state, long long *blkmin, void *state, const sfe_box *accepted,
                             const long long *n_accepted, sfe_box *act, cudaStream_t st);
int sfe_launch_spec_advance(void *state, const sfe_anchor *anchors, long long n, const long long *blkmin, long long K, long long span,
                            int esc_max, int tol, long long gap, int lookback, const uint8_t *cls, uint8_t *ext_state, sfe_box *act, int min_score, sfe_box *accepted,
                            long long accepted_cap, long long *win_idx, sfe_anchor *win_anchors, uint8_t *win_prio, uint8_t *keep,
                            sfe_result *results, sfe_stats *stats, const int32_t *plist, const uint8_t *lead_prio, cudaStream_t st);
int sfe_launch_spec_store(const sfe_result *wres, const long long *win_idx, long long wn, sfe_result *results, uint8_t *ext_state,
                          cudaStream_t st);
int sfe_launch_specl_finish(const void *state, long long *n_accepted_io, cudaStream_t st);
int sfe_launch_spec_promote(const sfe_result *wres, const long long *win_idx, long long wn, const sfe_anchor *anchors, long long n,
                            int min_score, int tol, long long reach, int max_ahead, const uint8_t *ext_state, uint8_t *cls, void *state,
                            int32_t *plist, cudaStream_t st);
int sfe_launch_len_bins(const sfe_result *res, long long n, uint8_t *prio, cudaStream_t st);
int sfe_launch_select_overflow(const sfe_half *halves, long long n_anchors, long long *sel, int32_t *tickets,
                               unsigned long long *counters, int n_chunks, cudaStream_t st);
int sfe_launch_probe(int mix, int iters, int blocks, int *sink, cudaStream_t st);
int sfe_launch_spec_prepare(const sfe_anchor *anchors, long long n, long long *blkmin, void *state, const sfe_box *accepted,
                            const long long *n_accepted, sfe_box *act, cudaStream_t st);
int sfe_launch_spec_scan(void *state, const sfe_anchor *anchors, long long n, const long long *blkmin, long long K, sfe_box *act,
                         long long *win_idx, sfe_anchor *win_anchors, uint8_t *keep, sfe_result *results, sfe_stats *stats,
                         cudaStream_t st);
int sfe_launch_spec_commit(void *state, const sfe_anchor *win_anchors, const sfe_result *wres, const long long *win_idx,
                           const long long *blkmin, int min_score, sfe_box *accepted, long long accepted_cap, sfe_box *act,
                           sfe_box *local, uint8_t *keep, sfe_result *results, sfe_stats *stats, cudaStream_t st);
int sfe_launch_spec_finish(const void *state, long long *n_accepted_io, cudaStream_t st);
int sfe_launch_spec_gather_kept(const sfe_anchor *anchors, const uint8_t *keep, long long n, sfe_anchor *kept_anchors,
                                long long *kept_idx, long long *n_kept, cudaStream_t st);
int sfe_launch_spec_scatter_kept(const sfe_result *kres, const long long *kept_idx, long long nk, sfe_result *results, cudaStream_t st);
int sfe_launch_ring_init(int32_t *ring, SfeFreeRing *st, int n_chunks, cudaStream_t stream);
int sfe_ydrop_init_device(void);

struct DevBuf {                       // grow-only device scratch
    void *p = nullptr; size_t cap = 0;
    int ensure(size_t bytes)
    {
        if (bytes <= cap) return SFE_OK;
        if (p) cudaFree(p);
        p = nullptr; cap = 0;
        size_t want = bytes + bytes / 4 + 256;
        if (cudaMalloc(&p, want) != cudaSuccess) { cudaGetLastError(); return SFE_ENOMEM; }
        cap = want;
        return SFE_OK;
    }
    void release() { if (p) cudaFree(p); p = nullptr; cap = 0; }
};

struct sfe_ctx {
    int device; cudaStream_t stream; int n_sm; int clock_khz;
    uint32_t *pool; int32_t *chunk_prev; int32_t *free_ring; SfeFreeRing *ring_state; int n_chunks;
    unsigned long long *counters;     // device, CNT_N
    unsigned long long *counters_host;  // pinned
    DevBuf halves, tickets, sel, hist, blkmin, act, misc, wide_tickets, long_tickets, wide_ring, ops_stage;
    DevBuf sp_state, sp_idx, sp_anchors, sp_results, sp_local, sp_blkmin, sp_act, sp_kanchors, sp_kidx, sp_kres;   // sfe_speculate
    DevBuf sp_cls, sp_ext, sp_prio, sp_plist, sp_lprio;   // predicted leaders
    long long opt[SFE_OPT_N];         // sfe_set_option
    long long spec_info[8];           // sfe_last_speculate_info
    long long *state_host;            // pinned, 16 words
    // host-API staging
    DevBuf h_tascii, h_qascii, h_t2, h_tm, h_q2, h_qm, h_r2, h_rm, h_pairs, h_anchors, h_results, h_keep, h_cigar, h_acc, h_small;
    long long info[SFE_INFO_N]; long long n_profile;
    cudaEvent_t ev0, ev1; bool ev_pending;
    cudaStream_t aux; cudaEvent_t ev_fork, ev_join;     // the cooperative row kernel runs beside the systolic one
    double kernel_us;
};

thread_local long long sfe_tls_launches = 0;
extern "C" int64_t sfe_launch_counter(void) { return (int64_t)sfe_tls_launches; }

static thread_local char g_err_detail[512] = "";      // per host thread: contexts driven from different threads do not race
void sfe_note_cuda_error(cudaError_t e, const char *file, int line)
{
    snprintf(g_err_detail, sizeof g_err_detail, "%s:%d: %s", file, line, cudaGetErrorString(e));
    cudaGetLastError();
}
void sfe_note_error_text(const char *msg) { snprintf(g_err_detail, sizeof g_err_detail, "%s", msg); }
extern "C" const char *sfe_last_error_detail(void) { return g_err_detail; }

static void harvest_kernel_time(sfe_ctx *c);

static const char *const k_errs[] = {"ok", "invalid argument", "out of memory", "CUDA error", "value outside supported range"};

extern "C" const char *sfe_strerror(int code)
{
    const int k = -code;
    return (k >= 0 && k <= 4) ? k_errs[k] : "unknown error";
}

extern "C" int sfe_create(sfe_ctx **out, int device, void *cuda_stream, size_t scratch_bytes)
{
    if (!out || device < 0) return SFE_EINVAL;
    *out = nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device >= ndev) { cudaGetLastError(); return SFE_ECUDA; }
    SFE_CUDA_CHECK(cudaSetDevice(device));
    cudaDeviceProp prop;
    SFE_CUDA_CHECK(cudaGetDeviceProperties(&prop, device));
    if (prop.major < 10) return SFE_ECUDA;                     // sm_100a only
    sfe_ctx *c = new (std::nothrow) sfe_ctx();
    if (!c) return SFE_ENOMEM;
    c->device = device; c->stream = (cudaStream_t)cuda_stream; c->n_sm = prop.multiProcessorCount;
    int khz = 0; cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, device); c->clock_khz = khz;
    if (scratch_bytes == 0) scratch_bytes = (size_t)1 << 30;
    long long nch = (long long)(scratch_bytes / SFE_CHUNK_BYTES);
    if (nch < 4) nch = 4;
    if (nch > 0x7ffffff0LL / SFE_CHUNK_RECS) nch = 0x7ffffff0LL / SFE_CHUNK_RECS;   // record indices are int32
    c->n_chunks = (int)nch;
    c->pool = nullptr; c->chunk_prev = nullptr; c->free_ring = nullptr; c->ring_state = nullptr; c->counters = nullptr; c->counters_host = nullptr; c->state_host = nullptr;
    memset(c->info, 0, sizeof c->info);
    memset(c->spec_info, 0, sizeof c->spec_info);
    c->opt[SFE_OPT_LEADER_DIAG_TOL] = 48; c->opt[SFE_OPT_LEADER_GAP] = 2000; c->opt[SFE_OPT_LEADER_LOOKBACK] = 64;
    c->opt[SFE_OPT_LEADER_NBREAK] = 64; c->opt[SFE_OPT_SPEC_SPAN] = 1 << 20; c->opt[SFE_OPT_SPEC_ESC_MAX] = 64;
    c->opt[SFE_OPT_SPARSE_WARPS] = 0; c->opt[SFE_OPT_FORCE_CLASS] = 0; c->opt[SFE_OPT_PROMOTE_REACH] = 65536; c->opt[SFE_OPT_ROW_KERNEL_CAP] = c->n_sm; c->opt[SFE_OPT_ROW_KERNEL_SCORE_ONLY] = 1;
    c->opt[SFE_OPT_LONG_ROWS] = 0; c->opt[SFE_OPT_LONG_ROWS_DENSE] = 0; c->opt[SFE_OPT_ROW_SLOTS] = 64;
    c->ev_pending = false; c->kernel_us = 0.0; c->n_profile = 0;
    if (cudaEventCreate(&c->ev0) != cudaSuccess || cudaEventCreate(&c->ev1) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming) != cudaSuccess ||
        cudaStreamCreateWithFlags(&c->aux, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); delete c; return SFE_ECUDA; }
    if (cudaMalloc((void **)&c->pool, (size_t)nch * SFE_CHUNK_BYTES) != cudaSuccess ||
        cudaMalloc((void **)&c->chunk_prev, (size_t)nch * sizeof(int32_t)) != cudaSuccess ||
        cudaMalloc((void **)&c->free_ring, (size_t)nch * sizeof(int32_t)) != cudaSuccess ||
        cudaMalloc((void **)&c->ring_state, sizeof(SfeFreeRing)) != cudaSuccess ||
        cudaMalloc((void **)&c->counters, CNT_N * sizeof(unsigned long long)) != cudaSuccess ||
        cudaMallocHost((void **)&c->counters_host, CNT_N * sizeof(unsigned long long)) != cudaSuccess ||
        cudaMallocHost((void **)&c->state_host, 16 * sizeof(long long)) != cudaSuccess) {
        cudaGetLastError();
        sfe_destroy(c);
        return SFE_ENOMEM;
    }
    if (sfe_launch_ring_init(c->free_ring, c->ring_state, c->n_chunks, c->stream) != SFE_OK) { sfe_destroy(c); return SFE_ECUDA; }
    if (sfe_ydrop_init_device() != SFE_OK) { sfe_destroy(c); return SFE_ECUDA; }      // function attributes are per device
    *out = c;
    return SFE_OK;
}

extern "C" int sfe_destroy(sfe_ctx *c)
{
    if (!c) return SFE_EINVAL;
    cudaSetDevice(c->device);
    if (c->pool) cudaFree(c->pool);
    if (c->chunk_prev) cudaFree(c->chunk_prev);
    if (c->free_ring) cudaFree(c->free_ring);
    if (c->ring_state) cudaFree(c->ring_state);
    if (c->counters) cudaFree(c->counters);
    if (c->counters_host) cudaFreeHost(c->counters_host);
    if (c->state_host) cudaFreeHost(c->state_host);
    cudaEventDestroy(c->ev0); cudaEventDestroy(c->ev1); cudaEventDestroy(c->ev_fork); cudaEventDestroy(c->ev_join);
    if (c->aux) { cudaStreamSynchronize(c->aux); cudaStreamDestroy(c->aux); }
    DevBuf *bufs[] = {&c->sp_cls, &c->sp_ext, &c->sp_prio, &c->sp_plist, &c->sp_lprio, &c->sp_kanchors, &c->sp_kidx, &c->sp_kres, &c->sp_state, &c->sp_idx, &c->sp_anchors, &c->sp_results, &c->sp_local, &c->sp_blkmin, &c->sp_act, &c->ops_stage, &c->wide_tickets, &c->long_tickets, &c->wide_ring, &c->halves, &c->tickets, &c->sel, &c->hist, &c->blkmin, &c->act, &c->misc, &c->h_tascii, &c->h_qascii,
                      &c->h_t2, &c->h_tm, &c->h_q2, &c->h_qm, &c->h_r2, &c->h_rm, &c->h_pairs, &c->h_anchors, &c->h_results,
                      &c->h_keep, &c->h_cigar, &c->h_acc, &c->h_small};
    for (DevBuf *b : bufs) b->release();
    delete c;
    return SFE_OK;
}

extern "C" int sfe_pack(sfe_ctx *c, const char *ascii_dev, int64_t len, uint8_t *codes2_dev, uint8_t *nmask_dev,
                        uint8_t *rc_codes2_dev, uint8_t *rc_nmask_dev)
{
    if (!c || len < 0 || (len > 0 && (!ascii_dev || !codes2_dev || !nmask_dev))) return SFE_EINVAL;
    if ((rc_codes2_dev == nullptr) != (rc_nmask_dev == nullptr)) return SFE_EINVAL;
    SFE_CUDA_CHECK(cudaSetDevice(c->device));
    return sfe_launch_pack(ascii_dev, len, codes2_dev, nmask_dev, rc_codes2_dev, rc_nmask_dev, c->stream);
}

extern "C" int sfe_probe_int_issue(sfe_ctx *c, int mix, int iters, double *lane_ops_per_clk_per_sm, double *elapsed_ms)
{
    if (!c || iters < 1 || mix < 0 || mix > 3 || !lane_ops_per_clk_per_sm) return SFE_EINVAL;
    SFE_CUDA_CHECK(cudaSetDevice(c->device));
    int rc = c->misc.ensure(256);
    if (rc) return rc;
    const int blocks = c->n_sm * 8;                            // 8 x 256 threads = 64 warps per SM
    cudaEvent_t e0, e1;
    SFE_CUDA_CHECK(cudaEventCreate(&e0)); SFE_CUDA_CHECK(cudaEventCreate(&e1));
    rc = sfe_launch_probe(mix, iters / 8 + 1, blocks, (int *)c->misc.p, c->stream);   // warm-up
    if (rc) return rc;
    SFE_CUDA_CHECK(cudaEventRecord(e0, c->stream));
    rc = sfe_launch_probe(mix, iters, blocks, (int *)c->misc.p, c->stream);
    if (rc) return rc;
    SFE_CUDA_CHECK(cudaEventRecord(e1, c->stream));
    SFE_CUDA_CHECK(cudaEventSynchronize(e1));
    float ms = 0.f;
    SFE_CUDA_CHECK(cudaEventElapsedTime(&ms, e0, e1));
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    // 16 instructions per thread per iteration (8 chains x 2 ops); the clock is sampled by the
    // caller (nvidia-smi) -- here we report per max-clock cycle and the elapsed time.
    const double lane_ops = (double)blocks * 256.0 * (double)iters * 16.0;
    const double cycles = (double)ms * 1e-3 * (double)c->clock_khz * 1e3;
    *lane_ops_per_clk_per_sm = lane_ops / cycles / (double)c->n_sm;
    if (elapsed_ms) *elapsed_ms = ms;
    return SFE_OK;
}

extern "C" int sfe_set_option(sfe_ctx *c, int key, int64_t value)
{
    if (!c || key < 0 || key >= SFE_OPT_N || value < 0) return SFE_EINVAL;
    if ((key == SFE_OPT_SPEC_SPAN || key == SFE_OPT_SPEC_ESC_MAX || key == SFE_OPT_LEADER_LOOKBACK) && value < 1) return SFE_EINVAL;
    if (key == SFE_OPT_SPARSE_WARPS && value > 16) return SFE_EINVAL;
    if (key == SFE_OPT_FORCE_CLASS && value > 3) return SFE_EINVAL;
    c->opt[key] = (long long)value;
    return SFE_OK;
}

extern "C" int sfe_last_speculate_info(sfe_ctx *c, int64_t info[8])
{
    if (!c || !info) return SFE_EINVAL;
    for (int k = 0; k < 8; k++) info[k] = c->spec_info[k];
    return SFE_OK;
}

extern "C" int sfe_last_batch_info(sfe_ctx *c, int64_t info[SFE_INFO_N])
{
    if (!c || !info) return SFE_EINVAL;
    harvest_kernel_time(c);
    c->info[6] = (long long)(c->kernel_us + 0.5);
    if (c->info[4] == 0) {   // score-only batches do not read the counters back inside the call
        if (cudaMemcpyAsync(c->counters_host, c->counters, CNT_N * sizeof(unsigned long long), cudaMemcpyDeviceToHost, c->stream) == cudaSuccess &&
            cudaStreamSynchronize(c->stream) == cudaSuccess) { c->info[4] = (long long)c->counters_host[CNT_STEPS]; c->info[5] = (long long)c->counters_host[CNT_WIDE]; c->info[7] = (long long)c->counters_host[CNT_BLOCK_HALVES]; c->info[8] = (long long)c->counters_host[CNT_RING_DROPS]; }
        else cudaGetLastError();
    }
    for (int k = 0; k < SFE_INFO_N; k++) info[k] = c->info[k];
    return SFE_OK;
}

extern "C" int sfe_last_half_profile(sfe_ctx *c, int64_t n, sfe_half_profile *out)
{
    if (!c || n < 0 || (n > 0 && !out)) return SFE_EINVAL;
    if (n > c->n_profile) n = c->n_profile;
    if (n == 0) return SFE_OK;
    SFE_CUDA_CHECK(cudaSetDevice(c->device));
    sfe_half *h = (sfe_half *)malloc((size_t)n * sizeof(sfe_half));
    if (!h) return SFE_ENOMEM;
    if (cudaMemcpyAsync(h, c->halves.p, (size_t)n * sizeof(sfe_half), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess ||
        cudaStreamSynchronize(c->stream) != cudaSuccess) { cudaGetLastError(); free(h); return SFE_ECUDA; }
    for (int64_t k = 0; k < n; k++) {
        out[k].cells = (int64_t)h[k].cells; out[k].cycles = h[k].cycles; out[k].steps = h[k].steps;
        out[k].n_strips = h[k].n_strips; out[k].max_steps = h[k].max_steps; out[k].n_ops = h[k].n_ops;
        out[k].smid = h[k].smid; out[k].wslot = h[k].wslot; out[k].status = h[k].status; out[k].reserved = 0;
    }
    free(h);
    return SFE_OK;
}

// add the device time of the last timed ydrop launch to kernel_us (needs the stream to have passed ev1)
static void harvest_kernel_time(sfe_ctx *c)
{
    if (!c->ev_pending) return;
    float ms = 0.f;
    if (cudaEventSynchronize(c->ev1) == cudaSuccess && cudaEventElapsedTime(&ms, c->ev0, c->ev1) == cudaSuccess) c->kernel_us += 1e3 * (double)ms;
    else cudaGetLastError();
    c->ev_pending = false;
}

// The row-synchronous block kernel (cooperative warps per half, f2) takes the pass only when asked to: it is
// bit-exact but, at one thread per window column, still slower per extension than the systolic chain.
static bool pick_block_kernel(const sfe_ctx *, long long, uint32_t flags)
{
    return (flags & SFE_BLOCK_KERNEL) != 0 && (flags & SFE_NO_BLOCK_KERNEL) == 0;
}

static int timed_ydrop(sfe_ctx *c, const YdParams &p, bool want_tb, uint32_t flags)
{
    harvest_kernel_time(c);
    SFE_CUDA_CHECK(cudaEventRecord(c->ev0, c->stream));
    const int rc = sfe_launch_ydrop(p, want_tb, pick_block_kernel(c, p.n_tickets, flags), c->n_sm, c->stream, c->aux, c->ev_fork, c->ev_join);
    if (rc) return rc;
    SFE_CUDA_CHECK(cudaEventRecord(c->ev1, c->stream));
    c->ev_pending = true;
    return SFE_OK;
}

// prune_lag: 32 (every kernel) or 0 (exact serial-order pruning: the row-synchronous block kernel only)
static int check_scoring(const sfe_scoring *s, uint32_t flags)
{
    if (!s) return SFE_EINVAL;
    if (s->prune_lag != SFE_PRUNE_LAG && !(s->prune_lag == 0 && (flags & SFE_BLOCK_KERNEL) && !(flags & SFE_NO_BLOCK_KERNEL))) return SFE_EINVAL;
    for (int a = 0; a < 4; a++)
        for (int b = 0; b < 4; b++)
            if (s->sub[a][b] < -128 || s->sub[a][b] > 127) return SFE_ELIMIT;
    if (s->n_score < -128 || s->n_score > 127) return SFE_ELIMIT;
    if (s->gap_open < 0 || s->gap_extend < 1 || s->gap_open + (long long)s->gap_extend > 65535) return SFE_ELIMIT;
    if (s->ydrop != SFE_YDROP_INF && (s->ydrop < 0 || s->ydrop >= (1 << 28))) return SFE_ELIMIT;
    return SFE_OK;
}

// first_of_series: reset the pool cursor and the batch info; later batches of a series (sfe_speculate's
// windows) append their ops to the same pool and accumulate the info counters.
static int ydrop_batch_impl(sfe_ctx *c, const uint8_t *t_codes2, const uint8_t *t_nmask, int64_t t_len,
                            const uint8_t *q_codes2, const uint8_t *q_nmask, const uint8_t *qrc_codes2,
                            const uint8_t *qrc_nmask, int64_t q_len, const sfe_pair *pairs_dev, int32_t n_pairs,
                            const sfe_anchor *anchors_dev, int64_t n_anchors, const sfe_scoring *sc, uint32_t flags,
                            sfe_result *results_dev, uint32_t *cigar_pool_dev, int64_t cigar_pool_cap,
                            int64_t *cigar_pool_used_dev, bool first_of_series, const uint8_t *prio_dev = nullptr, int sparse_warps = 0)
{
    if (!c || n_anchors < 0 || t_len < 0 || q_len < 0 || n_pairs < 0) return SFE_EINVAL;
    int rc = check_scoring(sc, flags);
    if (rc) return rc;
    const bool want_tb = (flags & SFE_WANT_CIGAR) != 0;
    if (n_anchors > 0 && (!t_codes2 || !t_nmask || !q_codes2 || !q_nmask || !pairs_dev || !anchors_dev || !results_dev)) return SFE_EINVAL;
    if ((qrc_codes2 == nullptr) != (qrc_nmask == nullptr)) return SFE_EINVAL;
    if (want_tb && (!cigar_pool_dev || cigar_pool_cap < 0 || !cigar_pool_used_dev)) return SFE_EINVAL;
    if (2 * n_anchors > 0x7ffffff0LL) return SFE_ELIMIT;
    SFE_CUDA_CHECK(cudaSetDevice(c->device));
    if (first_of_series) {
        memset(c->info, 0, sizeof c->info);
        c->ev_pending = false; c->kernel_us = 0.0;
        if (cigar_pool_used_dev) SFE_CUDA_CHECK(cudaMemsetAsync(cigar_pool_used_dev, 0, sizeof(int64_t), c->stream));
    }
    if (n_anchors == 0) return SFE_OK;

    if ((rc = c->halves.ensure((size_t)(2 * n_anchors) * sizeof(sfe_half)))) return rc;
    if ((rc = c->tickets.ensure((size_t)(2 * n_anchors) * sizeof(int32_t)))) return rc;
    if ((rc = c->hist.ensure(128 * sizeof(unsigned int)))) return rc;
    if ((rc = c->wide_tickets.ensure((size_t)(2 * n_anchors) * sizeof(int32_t)))) return rc;
    if ((rc = c->long_tickets.ensure((size_t)(4 * n_anchors) * sizeof(int32_t)))) return rc;
    if ((rc = c->wide_ring.ensure((size_t)SFE_WIDE_WARPS * RingGeom<SFE_WIDE_RING_LOG2>::WARP_BYTES))) return rc;
    if (want_tb && (rc = c->sel.ensure((size_t)n_anchors * sizeof(long long)))) return rc;
    // ops arena: every staged op ends up in the caller's pool, plus two header words per segment
    // (one segment per SFE_WALK_OPS ops, at least one per half)
    const unsigned long long ops_cap = want_tb ? (unsigned long long)cigar_pool_cap + (unsigned long long)cigar_pool_cap / (SFE_WALK_OPS / 2) +
                                                     4ULL * (unsigned long long)n_anchors + 64ULL : 0ULL;
    if (ops_cap > 0xfffffff0ULL) return SFE_ELIMIT;               // segment offsets are 32-bit
    if (want_tb && (rc = c->ops_stage.ensure((size_t)ops_cap * sizeof(uint32_t)))) return rc;

    YdParams p;
    memset(&p, 0, sizeof p);
    p.t_codes = t_codes2; p.t_nmask = t_nmask; p.q_codes = q_codes2; p.q_nmask = q_nmask;
    p.qrc_codes = qrc_codes2; p.qrc_nmask = qrc_nmask; p.t_len = t_len; p.q_len = q_len;
    p.pairs = pairs_dev; p.anchors = anchors_dev; p.tickets = (const int32_t *)c->tickets.p; p.n_tickets = 2 * n_anchors; p.seg_tickets = (flags & SFE_NO_BINNING) ? 0 : 4LL * c->n_sm;
    p.counters = c->counters; p.halves = (sfe_half *)c->halves.p; p.pool = c->pool; p.chunk_prev = c->chunk_prev; p.free_ring = c->free_ring; p.ring_state = c->ring_state;
    p.n_chunks = want_tb ? c->n_chunks : 0; p.n_pairs = n_pairs; p.max_warps = 0x7fffffff; p.sparse_warps = sparse_warps;
    p.wide_ring = (char *)c->wide_ring.p; p.wide_tickets = (int32_t *)c->wide_tickets.p;
    {   // hand-off of long halves to the row kernel (Lambda = 32 only; not when the caller pinned the kernel choice or the
        // priority tickets already go to the row kernel)
        const long long lr = c->opt[first_of_series ? SFE_OPT_LONG_ROWS_DENSE : SFE_OPT_LONG_ROWS];      // (a batch of sfe_speculate is never the first of a series)
        const bool on = lr > 0 && c->opt[SFE_OPT_ROW_SLOTS] > 0 && !(flags & (SFE_BLOCK_KERNEL | SFE_NO_BLOCK_KERNEL)) &&
                        sc->prune_lag == SFE_PRUNE_LAG && !(c->opt[SFE_OPT_ROW_KERNEL_CAP] > 0 && prio_dev != nullptr);
        p.long_strips = 0;
        if (on) { long long st = 1; while (st * 32 < lr && st < (1 << 24)) st *= 2; p.long_strips = (int)st; }     // strips, a power of two
        p.row_slots = (int)(c->opt[SFE_OPT_ROW_SLOTS] < 1024 ? c->opt[SFE_OPT_ROW_SLOTS] : 1024);
        p.long_tickets = (int32_t *)c->long_tickets.p;
    }
    p.ops_stage = (uint32_t *)c->ops_stage.p; p.ops_cap = ops_cap;
    p.OX = sc->gap_open + sc->gap_extend; p.X = sc->gap_extend;
    p.lag0 = sc->prune_lag == 0;
    p.ydrop_inf = sc->ydrop == SFE_YDROP_INF; p.Y = p.ydrop_inf ? 0 : sc->ydrop;
    for (int a = 0; a < 4; a++) {
        uint32_t w = 0;
        for (int b = 0; b < 4; b++) w |= ((uint32_t)(uint8_t)(int8_t)sc->sub[a][b]) << (8 * b);
        p.srow[a] = w;
    }
    p.srow[4] = 0x01010101u * (uint32_t)(uint8_t)(int8_t)sc->n_score;
    p.srow_hi = (uint32_t)(uint8_t)(int8_t)sc->n_score | (0xE0u << 16);

    SFE_CUDA_CHECK(cudaMemsetAsync(c->counters, 0, CNT_N * sizeof(unsigned long long), c->stream));
    // the longest tickets go to the cooperative row kernel (one CTA per half) unless the caller pinned the kernel choice
    const bool row_split = !(flags & (SFE_BLOCK_KERNEL | SFE_NO_BLOCK_KERNEL | SFE_NO_BINNING)) && sc->prune_lag == SFE_PRUNE_LAG &&
                           c->opt[SFE_OPT_ROW_KERNEL_CAP] > 0 && prio_dev != nullptr && (want_tb || c->opt[SFE_OPT_ROW_KERNEL_SCORE_ONLY]);
    p.row_split = row_split ? 1 : 0;
    if ((rc = sfe_launch_tickets(anchors_dev, n_anchors, pairs_dev, n_pairs, q_len, !(flags & SFE_NO_BINNING), prio_dev,
                                 (unsigned int *)c->hist.p, (int32_t *)c->tickets.p, c->counters, row_split ? c->opt[SFE_OPT_ROW_KERNEL_CAP] : 0,
                                 0 /* proxy-binned tickets stay with the systolic kernel: beside a DENSE launch the row kernel's CTAs
                                      cost a third of the SM's systolic occupancy and run contended (C4: 64 -> 108 ms) */, c->stream))) return rc;
    if ((rc = timed_ydrop(c, p, want_tb, flags))) return rc;
    c->info[0] += 1; c->info[1] += 2 * n_anchors; c->n_profile = 2 * n_anchors;
    if ((rc = sfe_launch_join(anchors_dev, p.halves, n_anchors, nullptr, n_anchors, want_tb, results_dev, c->stream))) return rc;
    if (!want_tb) return SFE_OK;
    if ((rc = sfe_launch_scan_emit(p.halves, n_anchors, nullptr, n_anchors, p.ops_stage, results_dev, cigar_pool_dev,
                                   cigar_pool_cap, (long long *)cigar_pool_used_dev, c->stream))) return rc;

    // traceback-arena overflow: a half that found no free chunk finished score-only; every half returns its chunks
    // when it ends, so the arena is free again here: re-run the anchors that did not fit, among themselves
    long long prev_overflow = -1;
    for (;;) {
        SFE_CUDA_CHECK(cudaMemcpyAsync(c->counters_host, c->counters, CNT_N * sizeof(unsigned long long),
                                       cudaMemcpyDeviceToHost, c->stream));
        SFE_CUDA_CHECK(cudaStreamSynchronize(c->stream));
        c->info[3] += (long long)c->counters_host[CNT_TBBYTES];
        c->info[4] += (long long)c->counters_host[CNT_STEPS];
        c->info[5] += (long long)c->counters_host[CNT_WIDE];
        c->info[7] += (long long)c->counters_host[CNT_BLOCK_HALVES];
        c->info[8] += (long long)c->counters_host[CNT_RING_DROPS];
        const long long n_over = (long long)c->counters_host[CNT_OVERFLOW];
        if (n_over == 0) break;
        // no progress possible: the anchors that overflowed were already running alone
        if (prev_overflow >= 0 && n_over >= prev_overflow) break;
        prev_overflow = n_over;
        SFE_CUDA_CHECK(cudaMemsetAsync(c->counters, 0, CNT_N * sizeof(unsigned long long), c->stream));
        if ((rc = sfe_launch_select_overflow(p.halves, n_anchors, (long long *)c->sel.p, (int32_t *)c->tickets.p,
                                             c->counters, c->n_chunks, c->stream))) return rc;
        SFE_CUDA_CHECK(cudaMemcpyAsync(c->counters_host, c->counters, CNT_N * sizeof(unsigned long long),
                                       cudaMemcpyDeviceToHost, c->stream));
        SFE_CUDA_CHECK(cudaStreamSynchronize(c->stream));
        const long long n_sel = (long long)c->counters_host[CNT_RERUN];
        if (n_sel <= 0) break;
        p.n_tickets = 2 * n_sel;
        // admission: every admitted warp can get the chunks of the neediest half, so each pass completes halves
        const long long need = (long long)c->counters_host[CNT_MAXNEED] > 0 ? (long long)c->counters_host[CNT_MAXNEED] : 1;
        const long long admit = c->n_chunks / need;
        p.max_warps = (int)(admit < 1 ? 1 : (admit > 0x7fffffffLL ? 0x7fffffffLL : admit));
        if ((rc = timed_ydrop(c, p, true, flags))) return rc;
        c->info[0] += 1; c->info[1] += 2 * n_sel; c->info[2] += 2 * n_sel;
        if ((rc = sfe_launch_join(anchors_dev, p.halves, n_anchors, (const long long *)c->sel.p, n_sel, 1, results_dev, c->stream))) return rc;
        if ((rc = sfe_launch_scan_emit(p.halves, n_anchors, (const long long *)c->sel.p, n_sel, p.ops_stage, results_dev,
                                       cigar_pool_dev, cigar_pool_cap, (long long *)cigar_pool_used_dev, c->stream))) return rc;
    }
    return SFE_OK;
}

extern "C" int sfe_ydrop_batch(sfe_ctx *c, const uint8_t *t_codes2, const uint8_t *t_nmask, int64_t t_len,
                               const uint8_t *q_codes2, const uint8_t *q_nmask, const uint8_t *qrc_codes2,
                               const uint8_t *qrc_nmask, int64_t q_len, const sfe_pair *pairs_dev, int32_t n_pairs,
                               const sfe_anchor *anchors_dev, int64_t n_anchors, const sfe_scoring *sc, uint32_t flags,
                               sfe_result *results_dev, uint32_t *cigar_pool_dev, int64_t cigar_pool_cap,
                               int64_t *cigar_pool_used_dev)
{
    return ydrop_batch_impl(c, t_codes2, t_nmask, t_len, q_codes2, q_nmask, qrc_codes2, qrc_nmask, q_len, pairs_dev, n_pairs,
                            anchors_dev, n_anchors, sc, flags, results_dev, cigar_pool_dev, cigar_pool_cap, cigar_pool_used_dev, true);
}

extern "C" int sfe_speculate(sfe_ctx *c, const uint8_t *t_codes2, const uint8_t *t_nmask, int64_t t_len,
                             const uint8_t *q_codes2, const uint8_t *q_nmask, const uint8_t *qrc_codes2,
                             const uint8_t *qrc_nmask, int64_t q_len, const sfe_pair *pairs_dev, int32_t n_pairs,
                             const sfe_anchor *anchors_dev, int64_t n_anchors, const sfe_scoring *sc, uint32_t flags,
                             int64_t window_k, sfe_result *results_dev, uint8_t *keep_dev, uint32_t *cigar_pool_dev,
                             int64_t cigar_pool_cap, int64_t *cigar_pool_used_dev, sfe_box *accepted_dev,
                             int64_t accepted_cap, int64_t *n_accepted_dev, sfe_stats *stats_dev)
{
    if (!c || n_anchors < 0 || window_k < 1 || accepted_cap < 0) return SFE_EINVAL;
    int rc = check_scoring(sc, flags);
    if (rc) return rc;
    if (n_anchors > 0 && (!anchors_dev || !results_dev || !keep_dev || !accepted_dev || !n_accepted_dev)) return SFE_EINVAL;
    SFE_CUDA_CHECK(cudaSetDevice(c->device));
    memset(c->info, 0, sizeof c->info);
    c->ev_pending = false; c->kernel_us = 0.0;
    if (cigar_pool_used_dev) SFE_CUDA_CHECK(cudaMemsetAsync(cigar_pool_used_dev, 0, sizeof(int64_t), c->stream));
    if (n_anchors == 0) return SFE_OK;
    // SFE_CIGAR_KEPT_ONLY: the commit rule needs only score and box, and the score-only chain of a long extension is
    // 1.6x shorter -- speculate without pointers, then one traceback batch over the kept anchors (all in parallel)
    const bool kept_only = (flags & SFE_CIGAR_KEPT_ONLY) && (flags & SFE_WANT_CIGAR);
    const uint32_t flags2 = kept_only ? (flags & ~SFE_WANT_CIGAR) : flags;
    const long long K = window_k < n_anchors ? window_k : n_anchors;
    memset(c->spec_info, 0, sizeof c->spec_info);
    if (flags & SFE_SPEC_LEADERS) {
        // ---- Algorithm 3 with predicted leaders (resolve_kernel.cu): classify once, then advance / extend until done ----
        if (!t_nmask || !q_nmask) return SFE_EINVAL;
        if ((rc = c->sp_state.ensure(128)) || (rc = c->sp_idx.ensure((size_t)K * sizeof(long long))) ||
            (rc = c->sp_anchors.ensure((size_t)K * sizeof(sfe_anchor))) || (rc = c->sp_results.ensure((size_t)K * sizeof(sfe_result))) ||
            (rc = c->sp_prio.ensure((size_t)K)) || (rc = c->sp_cls.ensure((size_t)n_anchors + 8)) || (rc = c->sp_plist.ensure((size_t)n_anchors * sizeof(int32_t))) || (rc = c->sp_lprio.ensure((size_t)n_anchors)) || (rc = c->sp_ext.ensure((size_t)n_anchors)) ||
            (rc = c->sp_blkmin.ensure((size_t)((n_anchors + 31) / 32 + 32) * sizeof(long long))) ||
            (rc = c->sp_act.ensure((size_t)(n_anchors + accepted_cap + 1) * sizeof(sfe_box)))) return rc;
        long long *blkmin = (long long *)c->sp_blkmin.p;
        sfe_box *act = (sfe_box *)c->sp_act.p;
        uint8_t *cls = (uint8_t *)c->sp_cls.p, *ext = (uint8_t *)c->sp_ext.p;
        if ((rc = sfe_launch_specl_prepare(anchors_dev, n_anchors, t_nmask, t_len, q_nmask, qrc_nmask, q_len, (int)c->opt[SFE_OPT_LEADER_DIAG_TOL],
                                           c->opt[SFE_OPT_LEADER_GAP], (int)c->opt[SFE_OPT_LEADER_LOOKBACK], (int)c->opt[SFE_OPT_LEADER_NBREAK],
                                           cls, (uint8_t *)c->sp_lprio.p, ext, blkmin, c->sp_state.p, accepted_dev, (const long long *)n_accepted_dev, act, c->stream))) return rc;
        if (c->opt[SFE_OPT_FORCE_CLASS] == 1) SFE_CUDA_CHECK(cudaMemsetAsync(cls, 0, (size_t)n_anchors, c->stream));        // testing: nobody leads
        else if (c->opt[SFE_OPT_FORCE_CLASS] == 2) SFE_CUDA_CHECK(cudaMemsetAsync(cls, 1, (size_t)n_anchors, c->stream));   // everybody leads
        else if (c->opt[SFE_OPT_FORCE_CLASS] == 3) SFE_CUDA_CHECK(cudaMemsetAsync(cls + n_anchors / 2, 0, (size_t)(n_anchors - n_anchors / 2), c->stream));
        long long n_batches = 0;
        for (;;) {
            if ((rc = sfe_launch_spec_advance(c->sp_state.p, anchors_dev, n_anchors, blkmin, K, c->opt[SFE_OPT_SPEC_SPAN], (int)c->opt[SFE_OPT_SPEC_ESC_MAX],
                                              (int)c->opt[SFE_OPT_LEADER_DIAG_TOL], c->opt[SFE_OPT_LEADER_GAP], (int)c->opt[SFE_OPT_LEADER_LOOKBACK], cls, ext, act, sc->min_score, accepted_dev, accepted_cap, (long long *)c->sp_idx.p,
                                              (sfe_anchor *)c->sp_anchors.p, (uint8_t *)c->sp_prio.p, keep_dev, results_dev, stats_dev, (const int32_t *)c->sp_plist.p, (const uint8_t *)c->sp_lprio.p, c->stream))) return rc;
            SFE_CUDA_CHECK(cudaMemcpyAsync(c->state_host, c->sp_state.p, 13 * sizeof(long long), cudaMemcpyDeviceToHost, c->stream));
            SFE_CUDA_CHECK(cudaStreamSynchronize(c->stream));
            const long long cursor = c->state_host[0], wn = c->state_host[1];
            c->spec_info[0] = n_batches; c->spec_info[1] = c->state_host[9]; c->spec_info[2] = c->state_host[8]; c->spec_info[3] = c->state_host[10];
            c->spec_info[4] = c->state_host[12];
            if (wn <= 0) {
                if (cursor < n_anchors) return SFE_ECUDA;            // cannot happen: a stop always queues the anchor it stopped at
                break;
            }
            if ((rc = ydrop_batch_impl(c, t_codes2, t_nmask, t_len, q_codes2, q_nmask, qrc_codes2, qrc_nmask, q_len, pairs_dev, n_pairs,
                                       (const sfe_anchor *)c->sp_anchors.p, wn, sc, flags2, (sfe_result *)c->sp_results.p,
                                       cigar_pool_dev, cigar_pool_cap, cigar_pool_used_dev, false, (const uint8_t *)c->sp_prio.p,
                                       (int)c->opt[SFE_OPT_SPARSE_WARPS]))) return rc;
            harvest_kernel_time(c);
            if ((rc = sfe_launch_spec_store((const sfe_result *)c->sp_results.p, (const long long *)c->sp_idx.p, wn, results_dev, ext, c->stream))) return rc;
            if (c->opt[SFE_OPT_SPEC_ESC_MAX] > 1 && c->opt[SFE_OPT_FORCE_CLASS] == 0 &&
                (rc = sfe_launch_spec_promote((const sfe_result *)c->sp_results.p, (const long long *)c->sp_idx.p, wn, anchors_dev, n_anchors, sc->min_score,
                                              (int)c->opt[SFE_OPT_LEADER_DIAG_TOL], c->opt[SFE_OPT_PROMOTE_REACH], 8192, ext, cls, c->sp_state.p, (int32_t *)c->sp_plist.p, c->stream))) return rc;
            n_batches++;
        }
        if ((rc = sfe_launch_specl_finish(c->sp_state.p, (long long *)n_accepted_dev, c->stream))) return rc;
    } else {
    if ((rc = c->sp_state.ensure(64)) || (rc = c->sp_idx.ensure((size_t)K * sizeof(long long))) ||
        (rc = c->sp_anchors.ensure((size_t)K * sizeof(sfe_anchor))) || (rc = c->sp_results.ensure((size_t)K * sizeof(sfe_result))) ||
        (rc = c->sp_local.ensure((size_t)(K + 1) * sizeof(sfe_box))) ||
        (rc = c->sp_blkmin.ensure((size_t)((n_anchors + 31) / 32 + 32) * sizeof(long long))) ||
        (rc = c->sp_act.ensure((size_t)(n_anchors + accepted_cap + 1) * sizeof(sfe_box)))) return rc;
    long long *blkmin = (long long *)c->sp_blkmin.p;
    sfe_box *act = (sfe_box *)c->sp_act.p;
    if ((rc = sfe_launch_spec_prepare(anchors_dev, n_anchors, blkmin, c->sp_state.p, accepted_dev, (const long long *)n_accepted_dev,
                                      act, c->stream))) return rc;
    for (long long win = 0;; win++) {
        if ((rc = sfe_launch_spec_scan(c->sp_state.p, anchors_dev, n_anchors, blkmin, K, act, (long long *)c->sp_idx.p,
                                       (sfe_anchor *)c->sp_anchors.p, keep_dev, results_dev, stats_dev, c->stream))) return rc;
        SFE_CUDA_CHECK(cudaMemcpyAsync(c->state_host, c->sp_state.p, 5 * sizeof(long long), cudaMemcpyDeviceToHost, c->stream));
        SFE_CUDA_CHECK(cudaStreamSynchronize(c->stream));
        const long long wn = c->state_host[1];
        if (wn <= 0) break;
        if ((rc = ydrop_batch_impl(c, t_codes2, t_nmask, t_len, q_codes2, q_nmask, qrc_codes2, qrc_nmask, q_len, pairs_dev, n_pairs,
                                   (const sfe_anchor *)c->sp_anchors.p, wn, sc, flags2, (sfe_result *)c->sp_results.p,
                                   cigar_pool_dev, cigar_pool_cap, cigar_pool_used_dev, false))) return rc;
        harvest_kernel_time(c);
        if ((rc = sfe_launch_spec_commit(c->sp_state.p, (const sfe_anchor *)c->sp_anchors.p, (const sfe_result *)c->sp_results.p,
                                         (const long long *)c->sp_idx.p, blkmin, sc->min_score, accepted_dev, accepted_cap, act,
                                         (sfe_box *)c->sp_local.p, keep_dev, results_dev, stats_dev, c->stream))) return rc;
    }
    if ((rc = sfe_launch_spec_finish(c->sp_state.p, (long long *)n_accepted_dev, c->stream))) return rc;
    }
    if (!kept_only) return SFE_OK;
    if ((rc = c->sp_kanchors.ensure((size_t)n_anchors * sizeof(sfe_anchor))) || (rc = c->sp_kidx.ensure((size_t)n_anchors * sizeof(long long)))) return rc;
    long long *d_nk = (long long *)((char *)c->sp_state.p + 48);
    if ((rc = sfe_launch_spec_gather_kept(anchors_dev, keep_dev, n_anchors, (sfe_anchor *)c->sp_kanchors.p, (long long *)c->sp_kidx.p, d_nk, c->stream))) return rc;
    SFE_CUDA_CHECK(cudaMemcpyAsync(c->state_host, d_nk, sizeof(long long), cudaMemcpyDeviceToHost, c->stream));
    SFE_CUDA_CHECK(cudaStreamSynchronize(c->stream));
    const long long nk = c->state_host[0];
    if (nk <= 0) return SFE_OK;
    if ((rc = c->sp_kres.ensure((size_t)nk * sizeof(sfe_result))) || (rc = c->sp_prio.ensure((size_t)nk))) return rc;
    // The kept anchors' extensions are known (score-only): their tickets are binned by the TRUE span, longest first, and --
    // the pass being as long as its longest half -- run with the sparse residency of the leader batches.
    const bool lead = (flags & SFE_SPEC_LEADERS) != 0;
    if (lead) {
        if ((rc = sfe_launch_spec_scatter_kept(results_dev, (const long long *)c->sp_kidx.p, -nk, (sfe_result *)c->sp_kres.p, c->stream))) return rc;
        if ((rc = sfe_launch_len_bins((const sfe_result *)c->sp_kres.p, nk, (uint8_t *)c->sp_prio.p, c->stream))) return rc;
    }
    if ((rc = ydrop_batch_impl(c, t_codes2, t_nmask, t_len, q_codes2, q_nmask, qrc_codes2, qrc_nmask, q_len, pairs_dev, n_pairs,
                               (const sfe_anchor *)c->sp_kanchors.p, nk, sc, flags, (sfe_result *)c->sp_kres.p,
                               cigar_pool_dev, cigar_pool_cap, cigar_pool_used_dev, false, lead ? (const uint8_t *)c->sp_prio.p : nullptr,
                               lead ? (int)c->opt[SFE_OPT_SPARSE_WARPS] : 0))) return rc;
    harvest_kernel_time(c);
    return sfe_launch_spec_scatter_kept((const sfe_result *)c->sp_kres.p, (const long long *)c->sp_kidx.p, nk, results_dev, c->stream);
}

extern "C" int sfe_resolve(sfe_ctx *c, const sfe_anchor *anchors_dev, const sfe_result *results_dev, int64_t n,
                           int32_t min_score, sfe_box *accepted_dev, int64_t accepted_cap, int64_t *n_accepted_dev,
                           uint8_t *keep_dev, sfe_stats *stats_dev)
{
    if (!c || n < 0 || accepted_cap < 0) return SFE_EINVAL;
    if (n == 0) return SFE_OK;
    if (!anchors_dev || !keep_dev || !accepted_dev || !n_accepted_dev) return SFE_EINVAL;
    SFE_CUDA_CHECK(cudaSetDevice(c->device));
    int rc;
    if ((rc = c->blkmin.ensure((size_t)((n + 31) / 32 + 32) * sizeof(long long)))) return rc;
    if ((rc = c->act.ensure((size_t)(accepted_cap + 1) * sizeof(sfe_box)))) return rc;
    return sfe_launch_resolve(anchors_dev, results_dev, n, min_score, accepted_dev, accepted_cap, (long long *)n_accepted_dev,
                              keep_dev, stats_dev, (long long *)c->blkmin.p, (sfe_box *)c->act.p, c->stream);
}

// window_k <= 0: one speculative batch over all anchors + one resolve; window_k >= 1: sfe_speculate
static int extend_host_impl(sfe_ctx *c, const char *t_ascii, int64_t t_len, const char *q_ascii, int64_t q_len,
                            const sfe_pair *pairs, int32_t n_pairs, const sfe_anchor *anchors, int64_t n_anchors,
                            const sfe_scoring *sc, uint32_t flags, int64_t window_k, sfe_result *results_host, uint8_t *keep_host,
                            uint32_t *cigar_host, int64_t cigar_cap, int64_t *cigar_used_host, sfe_stats *stats_host)
{
    if (!c || !t_ascii || !q_ascii || !pairs || !anchors || !sc || !results_host || !keep_host) return SFE_EINVAL;
    if (t_len <= 0 || q_len <= 0 || n_pairs <= 0 || n_anchors <= 0) return SFE_EINVAL;
    const bool want_tb = (flags & SFE_WANT_CIGAR) != 0;
    if (want_tb && (!cigar_host || cigar_cap <= 0 || !cigar_used_host)) return SFE_EINVAL;
    SFE_CUDA_CHECK(cudaSetDevice(c->device));
    cudaStream_t st = c->stream;
    int rc;
    const size_t tb2 = ((size_t)(t_len + 3) / 4 + 15) & ~(size_t)15, tbm = ((size_t)(t_len + 7) / 8 + 15) & ~(size_t)15;
    const size_t qb2 = ((size_t)(q_len + 3) / 4 + 15) & ~(size_t)15, qbm = ((size_t)(q_len + 7) / 8 + 15) & ~(size_t)15;
    if ((rc = c->h_tascii.ensure((size_t)t_len + 16)) || (rc = c->h_qascii.ensure((size_t)q_len + 16)) ||
        (rc = c->h_t2.ensure(tb2)) || (rc = c->h_tm.ensure(tbm)) || (rc = c->h_q2.ensure(qb2)) || (rc = c->h_qm.ensure(qbm)) ||
        (rc = c->h_r2.ensure(qb2)) || (rc = c->h_rm.ensure(qbm)) || (rc = c->h_pairs.ensure((size_t)n_pairs * sizeof(sfe_pair))) ||
        (rc = c->h_anchors.ensure((size_t)n_anchors * sizeof(sfe_anchor))) ||
        (rc = c->h_results.ensure((size_t)n_anchors * sizeof(sfe_result))) || (rc = c->h_keep.ensure((size_t)n_anchors)) ||
        (rc = c->h_acc.ensure((size_t)(n_anchors + 1) * sizeof(sfe_box))) ||
        (rc = c->h_small.ensure(256)) || (want_tb && (rc = c->h_cigar.ensure((size_t)cigar_cap * sizeof(uint32_t)))))
        return rc;
    SFE_CUDA_CHECK(cudaMemcpyAsync(c->h_tascii.p, t_ascii, (size_t)t_len, cudaMemcpyHostToDevice, st));
    SFE_CUDA_CHECK(cudaMemcpyAsync(c->h_qascii.p, q_ascii, (size_t)q_len, cudaMemcpyHostToDevice, st));
    SFE_CUDA_CHECK(cudaMemcpyAsync(c->h_pairs.p, pairs, (size_t)n_pairs * sizeof(sfe_pair), cudaMemcpyHostToDevice, st));
    SFE_CUDA_CHECK(cudaMemcpyAsync(c->h_anchors.p, anchors, (size_t)n_anchors * sizeof(sfe_anchor), cudaMemcpyHostToDevice, st));
    SFE_CUDA_CHECK(cudaMemsetAsync(c->h_small.p, 0, 256, st));
    long long *d_used = (long long *)c->h_small.p;              // [0] cigar used, [1] n_accepted
    sfe_stats *d_stats = (sfe_stats *)((char *)c->h_small.p + 64);
    if ((rc = sfe_pack(c, (const char *)c->h_tascii.p, t_len, (uint8_t *)c->h_t2.p, (uint8_t *)c->h_tm.p, nullptr, nullptr))) return rc;
    if ((rc = sfe_pack(c, (const char *)c->h_qascii.p, q_len, (uint8_t *)c->h_q2.p, (uint8_t *)c->h_qm.p, (uint8_t *)c->h_r2.p,
                       (uint8_t *)c->h_rm.p))) return rc;
    if (window_k >= 1) {
        if ((rc = sfe_speculate(c, (uint8_t *)c->h_t2.p, (uint8_t *)c->h_tm.p, t_len, (uint8_t *)c->h_q2.p, (uint8_t *)c->h_qm.p,
                                (uint8_t *)c->h_r2.p, (uint8_t *)c->h_rm.p, q_len, (sfe_pair *)c->h_pairs.p, n_pairs,
                                (sfe_anchor *)c->h_anchors.p, n_anchors, sc, flags, window_k, (sfe_result *)c->h_results.p,
                                (uint8_t *)c->h_keep.p, (uint32_t *)c->h_cigar.p, cigar_cap, (int64_t *)d_used, (sfe_box *)c->h_acc.p,
                                n_anchors, (int64_t *)(d_used + 1), d_stats))) return rc;
    } else {
        if ((rc = sfe_ydrop_batch(c, (uint8_t *)c->h_t2.p, (uint8_t *)c->h_tm.p, t_len, (uint8_t *)c->h_q2.p, (uint8_t *)c->h_qm.p,
                                  (uint8_t *)c->h_r2.p, (uint8_t *)c->h_rm.p, q_len, (sfe_pair *)c->h_pairs.p, n_pairs,
                                  (sfe_anchor *)c->h_anchors.p, n_anchors, sc, flags, (sfe_result *)c->h_results.p,
                                  (uint32_t *)c->h_cigar.p, cigar_cap, (int64_t *)d_used))) return rc;
        if ((rc = sfe_resolve(c, (sfe_anchor *)c->h_anchors.p, (sfe_result *)c->h_results.p, n_anchors, sc->min_score,
                              (sfe_box *)c->h_acc.p, n_anchors, (int64_t *)(d_used + 1), (uint8_t *)c->h_keep.p, d_stats))) return rc;
    }
    SFE_CUDA_CHECK(cudaMemcpyAsync(results_host, c->h_results.p, (size_t)n_anchors * sizeof(sfe_result), cudaMemcpyDeviceToHost, st));
    SFE_CUDA_CHECK(cudaMemcpyAsync(keep_host, c->h_keep.p, (size_t)n_anchors, cudaMemcpyDeviceToHost, st));
    long long used = 0;
    if (want_tb) {
        SFE_CUDA_CHECK(cudaMemcpyAsync(&used, d_used, sizeof used, cudaMemcpyDeviceToHost, st));
        SFE_CUDA_CHECK(cudaStreamSynchronize(st));
        const long long ncopy = used < cigar_cap ? used : cigar_cap;
        if (ncopy > 0) SFE_CUDA_CHECK(cudaMemcpyAsync(cigar_host, c->h_cigar.p, (size_t)ncopy * sizeof(uint32_t), cudaMemcpyDeviceToHost, st));
        *cigar_used_host = used;
    }
    if (stats_host) SFE_CUDA_CHECK(cudaMemcpyAsync(stats_host, d_stats, sizeof(sfe_stats), cudaMemcpyDeviceToHost, st));
    SFE_CUDA_CHECK(cudaStreamSynchronize(st));
    return SFE_OK;
}

extern "C" int sfe_extend_host(sfe_ctx *c, const char *t_ascii, int64_t t_len, const char *q_ascii, int64_t q_len,
                               const sfe_pair *pairs, int32_t n_pairs, const sfe_anchor *anchors, int64_t n_anchors,
                               const sfe_scoring *sc, uint32_t flags, sfe_result *results_host, uint8_t *keep_host,
                               uint32_t *cigar_host, int64_t cigar_cap, int64_t *cigar_used_host, sfe_stats *stats_host)
{
    return extend_host_impl(c, t_ascii, t_len, q_ascii, q_len, pairs, n_pairs, anchors, n_anchors, sc, flags, 0, results_host,
                            keep_host, cigar_host, cigar_cap, cigar_used_host, stats_host);
}

extern "C" int sfe_speculate_host(sfe_ctx *c, const char *t_ascii, int64_t t_len, const char *q_ascii, int64_t q_len,
                                  const sfe_pair *pairs, int32_t n_pairs, const sfe_anchor *anchors, int64_t n_anchors,
                                  const sfe_scoring *sc, uint32_t flags, int64_t window_k, sfe_result *results_host,
                                  uint8_t *keep_host, uint32_t *cigar_host, int64_t cigar_cap, int64_t *cigar_used_host,
                                  sfe_stats *stats_host)
{
    if (window_k < 1) return SFE_EINVAL;
    return extend_host_impl(c, t_ascii, t_len, q_ascii, q_len, pairs, n_pairs, anchors, n_anchors, sc, flags, window_k,
                            results_host, keep_host, cigar_host, cigar_cap, cigar_used_host, stats_host);
}
