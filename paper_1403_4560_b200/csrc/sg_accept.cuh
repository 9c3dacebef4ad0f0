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

// ---- binary-search variant (Dims::bs_accept: every threshold of the codes c <= 6 is below 2^32, i.e. h != 0) ----
// k = #{c : r >= T_c} has the bits  k2 = [r >= T_3],  k1 = [r >= (k2 ? T_5 : T_1)],  k0 = [r >= T_(4 k2 + 2 k1)]
// because the thresholds are sorted: three compares instead of seven.  A compare is one carry-out addition
// (IADD3, ALU pipe) whose carry is turned into the mask G = all ones iff r >= T by one IMAD.X (FMA pipe); the
// threshold of the next level is selected arithmetically with IMADs (G is 0 or -1), also on the FMA pipe:
//   T_sel1 = T_1 + G2 (T_1 - T_5)
//   T_sel0 = T_0 + G1 (T_0 - T_2) + G2 [(T_0 - T_4) + G1 (T_0 - T_2 - T_4 + T_6)]
// ALU pipe: 3 per word-site instead of 7; FMA pipe: 8 instead of 10.  Exact for T in [0, 2^32) (T = 0: r >= 0
// always holds); T = 2^32 (h = 0: code 6) is not representable in 32 bits, hence the flag.
// Constants in SlotK: lo[0] = T_3, lo[1] = T_1, lo[2] = T_1 - T_5, lo[3] = T_0, lo[4] = T_0 - T_2, lo[5] = T_0 - T_4,
// lo[6] = T_0 - T_2 - T_4 + T_6 (all mod 2^32); b3c, nc, ec unused.
// nr = ~r.  The carry of nr + T is [T >= r + 1] = [r < T] for every T in [0, 2^32) (T = 0: never), so
// -1 + carry = all ones iff r >= T.  (A borrow-out subtraction would save the complement, but ptxas hands the
// hardware carry, not the PTX borrow, to a following madc; the add form has no such ambiguity.)
__device__ __forceinline__ uint32_t ge_mask(uint32_t nr, uint32_t T, uint32_t one, uint32_t mone)
{
    return cadd(nr, T, mone, one);
}

__device__ __forceinline__ void k_masks_bs(uint32_t r, const SlotK &K, uint32_t one, uint32_t mone, uint32_t &G2,
                                           uint32_t &G1, uint32_t &G0)
{
    const uint32_t nr = imad(r, mone, mone);                // -r - 1 = ~r, on the FMA pipe
    G2 = ge_mask(nr, K.lo[0], one, mone);
    G1 = ge_mask(nr, imad(G2, K.lo[2], K.lo[1]), one, mone);
    const uint32_t w = imad(G1, K.lo[4], K.lo[3]);
    const uint32_t x = imad(G1, K.lo[6], K.lo[5]);
    G0 = ge_mask(nr, imad(G2, x, w), one, mone);
}

// host / device helper: the seven BS constants from the seven sorted thresholds (each < 2^32)
__host__ __device__ inline void bs_constants(const uint32_t (&T)[7], uint32_t (&out)[7])
{
    out[0] = T[3];
    out[1] = T[1];
    out[2] = T[1] - T[5];
    out[3] = T[0];
    out[4] = T[0] - T[2];
    out[5] = T[0] - T[4];
    out[6] = T[0] - T[2] - T[4] + T[6];
}

// One word-site: count the unsatisfied bonds (n0 n1 n2), decide, return the accept word.
// ALU pipe: 8 (count) + 7 (carries; BS: 3) + 3 (comparator) + 1 (n2 | g2, folded into the flip by the caller).
template <bool BS>
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
    if constexpr (BS) {
        uint32_t G2, G1, G0;
        k_masks_bs(r, K, one, mone, G2, G1, G0);
        const uint32_t g0 = na | ~G0;
        const uint32_t g1 = lop3<LUT_GE>(n0, G1, g0);
        const uint32_t g2 = lop3<LUT_GE>(n1, G2, g1);
        return n2 | g2;
    } else {
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
}

// Same decision with the field alignment folded in (a = s ^ amask ^ 1...: na = ~(s ^ amask)) and the flip
// fused: returns the NEW spin word s ^ accept.  ALU pipe: 8 (count) + 7 (carries; BS: 3) + 4.
constexpr int LUT_G0 = (~((0xF0 ^ 0xCC) & 0xAA)) & 0xFF;                    // ~((a ^ b) & c) = na | ~c
template <bool BS>
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
    if constexpr (BS) {
        uint32_t G2, G1, G0;
        k_masks_bs(r, K, one, mone, G2, G1, G0);
        const uint32_t g0 = lop3<LUT_G0>(s, amask, G0);
        const uint32_t g1 = lop3<LUT_GE>(n0, G1, g0);
        const uint32_t g2 = lop3<LUT_GE>(n1, G2, g1);
        return lop3<LUT_FLIP>(s, n2, g2);
    } else {
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
}

// The ten SlotK words of slot constants from the 64-bit negated thresholds c64[c] = (uint64)(0 - thr[c]) of the
// seven sorted codes (SlotTab::c64): binary-search constants if BS, else the carry-chain ones (lo[7], b3c, nc, ec).
template <bool BS>
__host__ __device__ inline void slotk_words(const uint32_t (&c64lo)[7], const uint32_t (&c64hi)[7], uint32_t (&out)[10])
{
    if (BS) {
        uint32_t T[7], b[7];
        for (int c = 0; c < 7; ++c) T[c] = 0u - c64lo[c];          // thr < 2^32: thr = -(2^64 - thr) mod 2^32
        bs_constants(T, b);
        for (int c = 0; c < 7; ++c) out[c] = b[c];
        out[7] = out[8] = out[9] = 0u;
    } else {
        uint32_t zc[7];
        for (int c = 0; c < 7; ++c) {
            out[c] = c64lo[c];
            zc[c] = c64hi[c] == 0u ? 1u : 0u;                      // (0 - thr) as 64 bits: hi = 0 only for thr = 0
        }
        out[7] = zc[3] - 1u;
        out[8] = zc[1] + zc[5] - 1u;
        out[9] = zc[0] + zc[2] + zc[4] + zc[6] - 2u;
    }
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
