// Register-level pieces of the online softmax used by the tcgen05 attention kernels (Eq. 2,
// PAPER.md:42, evaluated with exp2 and log2(e)/sqrt(d) folded into the scale; R13).
//
// One thread owns one query row and holds NC consecutive logits of it in registers.  Packed f32x2
// FMA/ADD and the 3-input FMNMX halve the issue slots around the MUFU (16 ex2/clk/SM on B200,
// measured, whatever the operand width: DESIGN.md 7.2).  An FMA-pipe polynomial exp2 for part of
// the columns was measured slower in every mix and is not kept (A/B table).
#pragma once

#include <stdint.h>

#include "sm100_ptx.cuh"

namespace lvsa_sm {

using sm100::fast_exp2;
using sm100::pack_bf16x2;

__device__ __forceinline__ uint64_t pack2(float lo, float hi) {
    uint64_t r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(uint64_t v, float &lo, float &hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ uint64_t fma2(uint64_t a, uint64_t b, uint64_t c) {
    uint64_t r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ uint64_t add2(uint64_t a, uint64_t b) {
    uint64_t r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ float fmax3(float a, float b, float c) {
    float r;
    asm("max.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));
    return r;
}

// max over s[0..NC) with 3-input max, four independent chains.
template <int NC>
__device__ __forceinline__ float row_max(const float (&s)[NC]) {
    static_assert(NC % 32 == 0, "NC must be a multiple of 32");
    float m0 = fmax3(s[0], s[1], s[2]), m1 = fmax3(s[3], s[4], s[5]);
    float m2 = fmax3(s[6], s[7], s[8]), m3 = fmax3(s[9], s[10], s[11]);
    constexpr int START = 12, REST = NC - START;           // REST % 8 == 4
#pragma unroll
    for (int c = START; c + 8 <= NC; c += 8) {
        m0 = fmax3(m0, s[c], s[c + 1]); m1 = fmax3(m1, s[c + 2], s[c + 3]);
        m2 = fmax3(m2, s[c + 4], s[c + 5]); m3 = fmax3(m3, s[c + 6], s[c + 7]);
    }
    constexpr int TAIL = START + (REST / 8) * 8;            // 4 values left
    m0 = fmax3(m0, s[TAIL], s[TAIL + 1]);
    m1 = fmax3(m1, s[TAIL + 2], s[TAIL + 3]);
    return fmaxf(fmax3(m0, m1, m2), m3);
}

// p = exp2(s * scale_log2 - m_use) for 32 consecutive logits s[C0..C0+32), packed to 16 bf16x2
// words; lsum (two packed fp32 partial sums) accumulates the fp32 values of p.
template <int NC>
__device__ __forceinline__ void exp_chunk32(const float (&s)[NC], int c0, uint64_t scale2, uint64_t negm2,
                                            uint32_t (&pk)[16], uint64_t &lsum) {
#pragma unroll
    for (int x = 0; x < 16; ++x) {
        const uint64_t xv = fma2(pack2(s[c0 + 2 * x], s[c0 + 2 * x + 1]), scale2, negm2);
        float a, b;
        unpack2(xv, a, b);
        const float p0 = fast_exp2(a), p1 = fast_exp2(b);
        lsum = add2(lsum, pack2(p0, p1));
        pk[x] = pack_bf16x2(p0, p1);
    }
}

}  // namespace lvsa_sm
