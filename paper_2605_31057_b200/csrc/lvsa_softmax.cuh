// Register-level pieces of the online softmax used by the tcgen05 attention kernels (Eq. 2,
// PAPER.md:42, evaluated with exp2 and log2(e)/sqrt(d) folded into the scale; R13).
//
// One thread owns one query row and holds NC consecutive logits of it in registers.  The MUFU
// unit (16 ex2/clk/SM on B200) would cap the kernel at the tensor-pipe time, so a compile-time
// fraction of the exponentials is evaluated on the FMA pipe instead: Cody-Waite split
// x = n + f (n = floor(x), f in [0,1)), a degree-3 polynomial for 2^f, and n added to the
// exponent field.  Max relative error of the polynomial is 8.6e-5, far below the bf16 rounding
// of P (2^-9) that follows it.  Packed f32x2 FMA/ADD and the 3-input FMNMX halve the issue slots.
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
__device__ __forceinline__ uint64_t add2_rm(uint64_t a, uint64_t b) {   // round toward -inf
    uint64_t r;
    asm("add.rm.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ float fmax3(float a, float b, float c) {
    float r;
    asm("max.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));
    return r;
}

// 2^x for the two lanes of xv on the FMA/ALU pipes; x is clamped to >= -126 (2^-126 ~ 1e-38
// stands in for anything smaller, including exp2(-inf)).
__device__ __forceinline__ void poly_exp2_pair(uint64_t xv, float &p0, float &p1) {
    constexpr float MAGIC = 12582912.f;   // 1.5 * 2^23: x + MAGIC (round down) holds floor(x) in its low bits
    float a, b;
    unpack2(xv, a, b);
    a = fmaxf(a, -126.f);
    b = fmaxf(b, -126.f);
    const uint64_t xc = pack2(a, b);
    const uint64_t xf = add2_rm(xc, pack2(MAGIC, MAGIC));
    const uint64_t xr = add2(xf, pack2(-MAGIC, -MAGIC));                 // floor(x) as a float
    const uint64_t fr = fma2(xr, pack2(-1.f, -1.f), xc);                 // f = x - floor(x)
    uint64_t p = fma2(fr, pack2(0.07706601917743683f, 0.07706601917743683f),
                      pack2(0.2276461124420166f, 0.2276461124420166f));
    p = fma2(p, fr, pack2(0.6951165199279785f, 0.6951165199279785f));
    p = fma2(p, fr, pack2(1.f, 1.f));
    float q0, q1, f0, f1;
    unpack2(p, q0, q1);
    unpack2(xf, f0, f1);
    p0 = __int_as_float(__float_as_int(q0) + (__float_as_int(f0) << 23));
    p1 = __int_as_float(__float_as_int(q1) + (__float_as_int(f1) << 23));
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

// Whether pair x (0..15) of a 32-column chunk goes to the polynomial: POLY of every 16 pairs,
// spread evenly so MUFU and FMA work interleave in the instruction stream.
template <int POLY>
__device__ __forceinline__ constexpr bool pair_uses_poly(int x) {
    return POLY > 0 && ((x * POLY) % 16) < POLY;
}

// p = exp2(s * scale_log2 - m_use) for 32 consecutive logits s[C0..C0+32), packed to 16 bf16x2
// words; lsum (two packed fp32 partial sums) accumulates the fp32 values of p.
template <int POLY, int NC>
__device__ __forceinline__ void exp_chunk32(const float (&s)[NC], int c0, uint64_t scale2, uint64_t negm2,
                                            uint32_t (&pk)[16], uint64_t &lsum) {
#pragma unroll
    for (int x = 0; x < 16; ++x) {
        const uint64_t xv = fma2(pack2(s[c0 + 2 * x], s[c0 + 2 * x + 1]), scale2, negm2);
        float p0, p1;
#ifdef LVSA_DIAG_NOEXP   // timing diagnostic only (wrong results): no exponential at all
        unpack2(xv, p0, p1);
#else
        if (pair_uses_poly<POLY>(x)) {
            poly_exp2_pair(xv, p0, p1);
        } else {
            float a, b;
            unpack2(xv, a, b);
            p0 = fast_exp2(a);
            p1 = fast_exp2(b);
        }
#endif
        lsum = add2(lsum, pack2(p0, p1));
        pk[x] = pack_bf16x2(p0, p1);
    }
}

}  // namespace lvsa_sm
