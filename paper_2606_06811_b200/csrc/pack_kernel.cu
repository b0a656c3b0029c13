// pack_kernel.cu -- a1: ASCII -> 2-bit code plane + 1-bit N-mask plane (+ reverse-complement
// planes) (R13, R14).  Bandwidth-trivial: each thread turns 32 bases (two 128-bit loads when
// aligned) into 8 code bytes and 4 mask bytes.
#include "sfe_internal.cuh"

static __device__ __forceinline__ uint32_t ascii_code(uint32_t c)
{
    c &= 0xDFu;                                   // fold case
    return c == 'A' ? 0u : c == 'C' ? 1u : c == 'G' ? 2u : c == 'T' ? 3u : 4u;
}

// forward planes: thread x handles bases [32x, 32x+32)
__global__ void pack_fwd_kernel(const char *ascii, long long len, uint8_t *codes2, uint8_t *nmask)
{
    const long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    const long long k0 = x * 32;
    if (k0 >= len) return;
    unsigned long long code = 0; uint32_t mask = 0;
    if (k0 + 32 <= len && ((uintptr_t)(ascii + k0) & 15) == 0) {
        const uint4 v0 = *(const uint4 *)(ascii + k0), v1 = *(const uint4 *)(ascii + k0 + 16);
        const uint32_t w[8] = {v0.x, v0.y, v0.z, v0.w, v1.x, v1.y, v1.z, v1.w};
#pragma unroll
        for (int i = 0; i < 32; i++) {
            const uint32_t c = ascii_code((w[i >> 2] >> ((i & 3) * 8)) & 0xff);
            if (c > 3) mask |= 1u << i; else code |= (unsigned long long)c << (2 * i);
        }
    } else {
        for (int i = 0; i < 32 && k0 + i < len; i++) {
            const uint32_t c = ascii_code((uint8_t)ascii[k0 + i]);
            if (c > 3) mask |= 1u << i; else code |= (unsigned long long)c << (2 * i);
        }
    }
    const long long nb_c = (len + 3) / 4, nb_m = (len + 7) / 8;
    for (int b = 0; b < 8 && x * 8 + b < nb_c; b++) codes2[x * 8 + b] = (uint8_t)(code >> (8 * b));
    for (int b = 0; b < 4 && x * 4 + b < nb_m; b++) nmask[x * 4 + b] = (uint8_t)(mask >> (8 * b));
}

// reverse-complement planes: thread x produces rc bases [32x, 32x+32) = complement of
// ascii[len-1-32x], ascii[len-2-32x], ...
__global__ void pack_rc_kernel(const char *ascii, long long len, uint8_t *rc_codes2, uint8_t *rc_nmask)
{
    const long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    const long long k0 = x * 32;
    if (k0 >= len) return;
    unsigned long long code = 0; uint32_t mask = 0;
    for (int i = 0; i < 32 && k0 + i < len; i++) {
        const uint32_t c = ascii_code((uint8_t)ascii[len - 1 - (k0 + i)]);
        if (c > 3) mask |= 1u << i; else code |= (unsigned long long)(3u - c) << (2 * i);
    }
    const long long nb_c = (len + 3) / 4, nb_m = (len + 7) / 8;
    for (int b = 0; b < 8 && x * 8 + b < nb_c; b++) rc_codes2[x * 8 + b] = (uint8_t)(code >> (8 * b));
    for (int b = 0; b < 4 && x * 4 + b < nb_m; b++) rc_nmask[x * 4 + b] = (uint8_t)(mask >> (8 * b));
}

int sfe_launch_pack(const char *ascii, long long len, uint8_t *codes2, uint8_t *nmask, uint8_t *rc_codes2,
                    uint8_t *rc_nmask, cudaStream_t st)
{
    if (len <= 0) return SFE_OK;
    const long long nthreads = (len + 31) / 32;
    const int bs = 256;
    const unsigned nb = (unsigned)((nthreads + bs - 1) / bs);
    SFE_KL pack_fwd_kernel<<<nb, bs, 0, st>>>(ascii, len, codes2, nmask);
    if (rc_codes2 && rc_nmask) SFE_KL pack_rc_kernel<<<nb, bs, 0, st>>>(ascii, len, rc_codes2, rc_nmask);
    SFE_LAUNCH_CHECK();
}
