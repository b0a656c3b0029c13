// sfe_resolve_static: the resolve rule (a9; Alg. 3 phase 3; R16, R17, R26) for callers that must not
// allocate -- code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc.  It needs no sfe_ctx (sfe_create
// allocates) and calls no cudaMalloc / cudaFree / allocating library routine: the two scratch regions the resolve kernels
// use (the per-32-anchor minima of tpos with their suffix minimum, and the active-box list) live in ONE file-scope
// __device__ array of fixed size.  Every GPU that loads libsfe.so holds that array (2.75 MiB) until the process exits.
//
// In host code the array's name is a host-side stand-in, not a device address.  The address the kernels get comes from
// cudaGetSymbolAddress, asked once per device with that device current (static_scratch_base below).
//
// The kernels are the ones sfe_resolve launches (resolve_kernel.cu), given this scratch instead of the context's buffers,
// so the two entry points cannot drift apart; tests/test_zz_no_alloc.py compares them byte for byte.
//
// Sharing: every call on a device uses the same array.  Nothing in it has to start at zero -- the minima of all
// ceil(n / 32) blocks are written by block_min_kernel and the active list is written before it is read, in every call --
// so the contents a previous call left behind are never read.  Calls that overlap on the GPU (two streams, two host
// threads, two graphs replayed concurrently) race on it: serialise them on one stream or with events.
#include "sfe_internal.cuh"
#include <mutex>

// resolve_kernel.cu: block_min_kernel + resolve_kernel on the given scratch (blkmin: ceil(n / 32) + 32 entries; act: accepted_cap + 1 boxes)
int sfe_launch_resolve(const sfe_anchor *anchors, const sfe_result *results, long long n, int min_score, sfe_box *accepted,
                       long long accepted_cap, long long *n_accepted_io, uint8_t *keep, sfe_stats *stats, long long *blkmin,
                       sfe_box *act, cudaStream_t st);

#define STATIC_BLKMIN_BYTES ((((size_t)SFE_STATIC_MAX_ANCHORS / 32 + 32) * sizeof(long long) + 255) & ~(size_t)255)
#define STATIC_ACT_BYTES    ((((size_t)SFE_STATIC_MAX_ACCEPTED + 1) * sizeof(sfe_box) + 255) & ~(size_t)255)

static __device__ __align__(256) unsigned char g_resolve_scratch[STATIC_BLKMIN_BYTES + STATIC_ACT_BYTES];

#define STATIC_MAX_DEVICES 64
static std::mutex g_static_mu;
static unsigned char *g_static_base[STATIC_MAX_DEVICES];       // device address of g_resolve_scratch, per device (0: not asked yet)

// Set-up, once per device: `device` must be the current device.
static int static_scratch_base(int device, unsigned char **base)
{
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_base[device]) {
        unsigned char *p = nullptr;
        SFE_CUDA_CHECK(cudaGetSymbolAddress((void **)&p, g_resolve_scratch));
        if (!p) return SFE_ECUDA;
        g_static_base[device] = p;
    }
    *base = g_static_base[device];
    return SFE_OK;
}

extern "C" int sfe_resolve_static_limits(int64_t *max_anchors, int64_t *max_accepted, int64_t *scratch_bytes)
{
    if (max_anchors) *max_anchors = SFE_STATIC_MAX_ANCHORS;
    if (max_accepted) *max_accepted = SFE_STATIC_MAX_ACCEPTED;
    if (scratch_bytes) *scratch_bytes = (int64_t)sizeof g_resolve_scratch;
    return SFE_OK;
}

extern "C" int sfe_resolve_static(int device, void *cuda_stream, const sfe_anchor *anchors_dev, const sfe_result *results_dev,
                                  int64_t n, int32_t min_score, sfe_box *accepted_dev, int64_t accepted_cap,
                                  int64_t *n_accepted_dev, uint8_t *keep_dev, sfe_stats *stats_dev)
{
    if (device < 0 || device >= STATIC_MAX_DEVICES || n < 0 || accepted_cap < 0) return SFE_EINVAL;
    if (n > SFE_STATIC_MAX_ANCHORS) {
        sfe_note_error_text("sfe_resolve_static: n exceeds SFE_STATIC_MAX_ANCHORS (1048576); use sfe_resolve, or split the anchors "
                            "into consecutive calls that carry accepted_dev");
        return SFE_ELIMIT;
    }
    if (accepted_cap > SFE_STATIC_MAX_ACCEPTED) {
        sfe_note_error_text("sfe_resolve_static: accepted_cap exceeds SFE_STATIC_MAX_ACCEPTED (65536); use sfe_resolve");
        return SFE_ELIMIT;
    }
    if (n == 0) return SFE_OK;
    if (!anchors_dev || !keep_dev || !accepted_dev || !n_accepted_dev) return SFE_EINVAL;
    SFE_CUDA_CHECK(cudaSetDevice(device));
    unsigned char *base = nullptr;
    const int rc = static_scratch_base(device, &base);
    if (rc) return rc;
    return sfe_launch_resolve(anchors_dev, results_dev, n, min_score, accepted_dev, accepted_cap, (long long *)n_accepted_dev,
                              keep_dev, stats_dev, (long long *)base, (sfe_box *)(base + STATIC_BLKMIN_BYTES),
                              (cudaStream_t)cuda_stream);
}
