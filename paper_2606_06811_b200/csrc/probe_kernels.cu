// probe_kernels.cu -- measurement only: the integer-issue microbenchmark behind sfe_probe_int_issue,
// which supplies the R (lane-instructions per clock per SM) of the integer-issue roofline.  Not on the hot path.
#include "sfe_internal.cuh"

// ---- integer-issue microbenchmark ---------------------------------------------------------------------
// Register-only loops of independent chains, one kernel per opcode mix, at full occupancy.  Each
// iteration issues OPS instructions per thread (checked against cuobjdump: DESIGN.md "Roofline").
#define PROBE_CHAINS 8
template <int MIX>
__global__ void __launch_bounds__(256) probe_kernel(int iters, int seed, int *sink)
{
    int a[PROBE_CHAINS], b[PROBE_CHAINS];
#pragma unroll
    for (int c = 0; c < PROBE_CHAINS; c++) { a[c] = seed + threadIdx.x * (c + 1); b[c] = seed ^ (c * 77 + blockIdx.x); }
    const int k1 = seed | 1, k2 = seed + 3;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int c = 0; c < PROBE_CHAINS; c++) {
            if (MIX == 1) {            // ALU pipe only: SHF + LOP3 (an add.s32 would become IMAD.IADD on the FMA pipe)
                asm volatile("shf.l.wrap.b32 %0, %0, %1, 3;" : "+r"(a[c]) : "r"(b[c]));
                asm volatile("xor.b32 %0, %0, %1;" : "+r"(b[c]) : "r"(a[c]));
            } else if (MIX == 2) {     // DPX: VIADDMNMX + VIMNMX3
                a[c] = __viaddmax_s32(a[c], k1, b[c]);
                b[c] = __vimax3_s32(b[c], a[c], k2);
            } else if (MIX == 3) {     // FMA pipe: IMAD
                asm volatile("mad.lo.s32 %0, %0, %1, %2;" : "+r"(a[c]) : "r"(k1), "r"(b[c]));
                asm volatile("mad.lo.s32 %0, %0, %1, %2;" : "+r"(b[c]) : "r"(k2), "r"(a[c]));
            } else {                   // mixed: one ALU/DPX op + one IMAD (both pipes busy)
                a[c] = __viaddmax_s32(a[c], k1, b[c]);
                asm volatile("mad.lo.s32 %0, %0, %1, %2;" : "+r"(b[c]) : "r"(k2), "r"(a[c]));
            }
        }
    }
    int r = 0;
#pragma unroll
    for (int c = 0; c < PROBE_CHAINS; c++) r ^= a[c] ^ b[c];
    if (r == 0x7fffabcd) *sink = r;
}

int sfe_launch_probe(int mix, int iters, int blocks, int *sink, cudaStream_t st)
{
    switch (mix) {
    case 1: SFE_KL probe_kernel<1><<<blocks, 256, 0, st>>>(iters, 12345, sink); break;
    case 2: SFE_KL probe_kernel<2><<<blocks, 256, 0, st>>>(iters, 12345, sink); break;
    case 3: SFE_KL probe_kernel<3><<<blocks, 256, 0, st>>>(iters, 12345, sink); break;
    default: SFE_KL probe_kernel<0><<<blocks, 256, 0, st>>>(iters, 12345, sink); break;
    }
    SFE_LAUNCH_CHECK();
}
