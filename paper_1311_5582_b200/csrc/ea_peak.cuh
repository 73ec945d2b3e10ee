// ea_peak.cuh -- integer-pipe issue-rate microbenchmark: the
// roofline denominator for the sweep kernel is MEASURED, not taken from a datasheet.
// Streams of independent LOP3 (ALU pipe), IMAD (FMA pipe) and a 1:1 mix, 8 chains per thread.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace ea {

template <int MODE>   // 0: LOP3 only, 1: IMAD only, 2: alternating LOP3 / IMAD
__global__ void __launch_bounds__(256) k_int_peak(uint32_t *out, int iters, uint32_t a, uint32_t b)
{
    uint32_t x[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = threadIdx.x * 8u + i + a;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int rep = 0; rep < 8; ++rep) {
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                if (MODE == 0 || (MODE == 2 && (i & 1) == 0))
                    asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x[i]) : "r"(a), "r"(b));
                else
                    asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(x[i]) : "r"(a), "r"(b));
            }
        }
    }
    uint32_t s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s ^= x[i];
    if (s == 0x12345u) out[0] = s;   // never true in practice; keeps the chains alive
}

}  // namespace ea
