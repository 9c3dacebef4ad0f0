// sg_accept.cuh — the branch-free Metropolis acceptance of the shared-memory-resident +-J kernels
// (sg_ladder8.cu, sg_res32.cu): Philox with precomputed round keys, the carry-chain comparator
// (DESIGN.md §5 "acceptance without branches") and the bit-sliced two-operand adder.
#pragma once
#include "sg_device.cuh"

namespace sg {

__device__ __forceinline__ uint4 philox_rk8(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, const uint32_t (&rk)[20])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = xor3((uint32_t)(p1 >> 32), c1, rk[2 * r]);
        const uint32_t n2 = xor3((uint32_t)(p0 >> 32), c3, rk[2 * r + 1]);
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
    }
    return make_uint4(c0, c1, c2, c3);
}

// acc * one + [r + lo carries]: one IADD3 (carry out only, ALU pipe) + one IMAD.X (FMA pipe).  `one` is a
// run-time 1, so ptxas keeps the multiply-add-with-carry on the FMA pipe instead of an IADD3.X.
__device__ __forceinline__ uint32_t cadd(uint32_t r, uint32_t lo, uint32_t acc, uint32_t one)
{
    uint32_t d;
    asm("{\n\t.reg .u32 t;\n\tadd.cc.u32 t, %1, %2;\n\tmadc.lo.u32 %0, %3, %4, 0;\n\t}" : "=r"(d) : "r"(r), "r"(lo), "r"(acc), "r"(one));
    return d;
}

__device__ __forceinline__ uint32_t imad(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t d;
    asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}

// Per-slot acceptance constants: lo[c] = 2^32 - thr[c] (mod 2^32) for the 7 sorted
// non-trivial thresholds (code c = 2 n_u + (1-a)); the carry of r + lo[c] is C_c = [r >= thr[c]]
// (a threshold of 0 cannot carry: its C_c = 1 is folded into the chain start constants).
//   B3  = C_3 - 1                       all ones iff r <  thr[3]   (K2 = ~B3)
//   Nn  = C_1 + C_5 - 1
//   E   = C_0 + C_2 + C_4 + C_6 - 2
//   K1m = B3 - Nn        = -(k bit 1),  K0m = Nn + B3 - E = -(k bit 0),  k = #{c : r >= thr[c]}
// (exact because the thresholds are sorted: C_0 >= C_1 >= ... >= C_6).
struct SlotK {
    uint32_t lo[7];
    uint32_t b3c, nc, ec;
};

// One word-site: count the unsatisfied bonds (n0 n1 n2), decide, return the accept word.
// ALU pipe: 8 (count) + 7 (carries) + 3 (comparator) + 1 (n2 | g2, folded into the flip by the caller).
__device__ __forceinline__ uint32_t accept_word(uint32_t u0, uint32_t u1, uint32_t u2, uint32_t u3, uint32_t u4,
                                                uint32_t u5, uint32_t na, uint32_t r, const SlotK &K, uint32_t one,
                                                uint32_t mone, uint32_t &n0, uint32_t &n1, uint32_t &n2)
{
    const uint32_t s0 = xor3(u0, u1, u2), c0 = maj3(u0, u1, u2);
    const uint32_t s1 = xor3(u3, u4, u5), c1 = maj3(u3, u4, u5);
    n0 = s0 ^ s1;
    const uint32_t k = s0 & s1;
    n1 = xor3(c0, c1, k);
    n2 = maj3(c0, c1, k);
    const uint32_t B3 = cadd(r, K.lo[3], K.b3c, one);
    const uint32_t Nn = cadd(r, K.lo[5], cadd(r, K.lo[1], K.nc, one), one);
    const uint32_t E = cadd(r, K.lo[6], cadd(r, K.lo[4], cadd(r, K.lo[2], cadd(r, K.lo[0], K.ec, one), one), one), one);
    const uint32_t K1m = imad(Nn, mone, B3);
    const uint32_t K0m = imad(Nn, one, imad(E, mone, B3));
    const uint32_t g0 = na | ~K0m;
    const uint32_t g1 = lop3<LUT_GE>(n0, K1m, g0);
    const uint32_t g2 = lop3<LUT_MAJ>(n1, B3, g1);             // GE(n1, K2, g1) with K2 = ~B3
    return n2 | g2;
}

// Same decision with the field alignment folded in (a = s ^ amask ^ 1...: na = ~(s ^ amask)) and the flip
// fused: returns the NEW spin word s ^ accept.  ALU pipe: 8 (count) + 7 (carries) + 4.
constexpr int LUT_G0 = (~((0xF0 ^ 0xCC) & 0xAA)) & 0xFF;                    // ~((a ^ b) & c) = na | ~c
__device__ __forceinline__ uint32_t flip_word_k(uint32_t s, uint32_t amask, uint32_t u0, uint32_t u1, uint32_t u2,
                                                uint32_t u3, uint32_t u4, uint32_t u5, uint32_t r, const SlotK &K,
                                                uint32_t one, uint32_t mone)
{
    const uint32_t s0 = xor3(u0, u1, u2), c0 = maj3(u0, u1, u2);
    const uint32_t s1 = xor3(u3, u4, u5), c1 = maj3(u3, u4, u5);
    const uint32_t n0 = s0 ^ s1;
    const uint32_t k = s0 & s1;
    const uint32_t n1 = xor3(c0, c1, k);
    const uint32_t n2 = maj3(c0, c1, k);
    const uint32_t B3 = cadd(r, K.lo[3], K.b3c, one);
    const uint32_t Nn = cadd(r, K.lo[5], cadd(r, K.lo[1], K.nc, one), one);
    const uint32_t E = cadd(r, K.lo[6], cadd(r, K.lo[4], cadd(r, K.lo[2], cadd(r, K.lo[0], K.ec, one), one), one), one);
    const uint32_t K1m = imad(Nn, mone, B3);
    const uint32_t K0m = imad(Nn, one, imad(E, mone, B3));
    const uint32_t g0 = lop3<LUT_G0>(s, amask, K0m);
    const uint32_t g1 = lop3<LUT_GE>(n0, K1m, g0);
    const uint32_t g2 = lop3<LUT_MAJ>(n1, B3, g1);
    return lop3<LUT_FLIP>(s, n2, g2);
}

// bit-sliced a (NA planes) + b (NA planes) -> NA+1 planes
template <int NA>
__device__ __forceinline__ void bs_sum(const uint32_t (&a)[NA], const uint32_t (&b)[NA], uint32_t (&o)[NA + 1])
{
    uint32_t carry = a[0] & b[0];
    o[0] = a[0] ^ b[0];
#pragma unroll
    for (int k = 1; k < NA; ++k) {
        o[k] = xor3(a[k], b[k], carry);
        carry = maj3(a[k], b[k], carry);
    }
    o[NA] = carry;
}

}  // namespace sg
