// sg_device.cuh — device-side building blocks shared by the kernels of libsg_b200 (sm_100a).
//
// Philox4x32-10 (Salmon et al., SC'11), the written-IEEE-sequence elementary functions of
// DESIGN.md R12-R14, LOP3 helpers, bit-sliced adders and the 32x32 warp bit transpose.
// Nothing here is shared with oracle/ (which restates the same definitions in plain C).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace sg {

// ------------------------------------------------------------------------------------ LOP3
// 3-input boolean function with truth table LUT (a = 0xF0, b = 0xCC, c = 0xAA).
template <int LUT>
__device__ __forceinline__ uint32_t lop3(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t d;
    asm("lop3.b32 %0, %1, %2, %3, %4;" : "=r"(d) : "r"(a), "r"(b), "r"(c), "n"(LUT));
    return d;
}
constexpr int LUT_XOR3 = 0xF0 ^ 0xCC ^ 0xAA;                               // a ^ b ^ c
constexpr int LUT_MAJ = (0xF0 & 0xCC) | (0xCC & 0xAA) | (0xF0 & 0xAA);      // majority
constexpr int LUT_GE = (0xF0 & ~0xCC & 0xFF) | ((~(0xF0 ^ 0xCC)) & 0xAA & 0xFF); // (a&~b) | (~(a^b)&c)
constexpr int LUT_FLIP = 0xF0 ^ (0xCC | 0xAA);                              // a ^ (b | c)
constexpr int LUT_K1 = ((~0xF0 & 0xCC) | (~0xAA)) & 0xFF;                   // (~a & b) | ~c

__device__ __forceinline__ uint32_t xor3(uint32_t a, uint32_t b, uint32_t c) { return lop3<LUT_XOR3>(a, b, c); }
__device__ __forceinline__ uint32_t maj3(uint32_t a, uint32_t b, uint32_t c) { return lop3<LUT_MAJ>(a, b, c); }

// ------------------------------------------------------------------------- Philox4x32-10
// Round keys are k + round * (0x9E3779B9, 0xBB67AE85); 10 rounds; output = final counter.
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = xor3((uint32_t)(p1 >> 32), c1, k0);
        const uint32_t n2 = xor3((uint32_t)(p0 >> 32), c3, k1);
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    return make_uint4(c0, c1, c2, c3);
}

// counter word 3 of DESIGN.md R5
__device__ __forceinline__ uint32_t ctr3(uint32_t domain, uint32_t replica, uint32_t slot)
{
    return (domain << 24) | (replica << 16) | slot;
}

// ------------------------------------------------- written IEEE sequences (R12, R13, R14)
// Every multiply / add is a separately rounded IEEE operation (__dmul_rn etc. are never
// contracted); the library is also compiled with -fmad=false.

// 2^32 * exp(-y), rounded down, y > 0; tab[i] = exp(-i/256) (host libm), i <= 5760.
__device__ __forceinline__ uint64_t dexp64(const double *__restrict__ tab, double y)
{
    if (!(y < 22.5)) return 0;
    const int i = __double2int_rz(__dmul_rn(y, 256.0));
    const double f = __dsub_rn(y, __dmul_rn((double)i, 0.00390625));
    const double z = -f;
    double g = 0x1.6c16c16c16c17p-10;
    g = __dadd_rn(__dmul_rn(g, z), 0x1.1111111111111p-7);
    g = __dadd_rn(__dmul_rn(g, z), 0x1.5555555555555p-5);
    g = __dadd_rn(__dmul_rn(g, z), 0x1.5555555555555p-3);
    g = __dadd_rn(__dmul_rn(g, z), 0x1.0000000000000p-1);
    g = __dadd_rn(__dmul_rn(g, z), 1.0);
    g = __dadd_rn(__dmul_rn(g, z), 1.0);
    const double p = __dmul_rn(tab[i], g);
    return __double2ull_rz(__dmul_rn(p, 4294967296.0));
}

// fp32 analogue: step 1/64, degree 4; tab[i] = (float)exp(-i/64), i <= 1440.
__device__ __forceinline__ uint64_t dexp32(const float *__restrict__ tab, float y)
{
    if (!(y < 22.5f)) return 0;
    const int i = __float2int_rz(__fmul_rn(y, 64.0f));
    const float f = __fsub_rn(y, __fmul_rn((float)i, 0.015625f));
    const float z = -f;
    float g = 0x1.555556p-5f;
    g = __fadd_rn(__fmul_rn(g, z), 0x1.555556p-3f);
    g = __fadd_rn(__fmul_rn(g, z), 0.5f);
    g = __fadd_rn(__fmul_rn(g, z), 1.0f);
    g = __fadd_rn(__fmul_rn(g, z), 1.0f);
    const float p = __fmul_rn(tab[i], g);
    return __float2ull_rz(__fmul_rn(p, 4294967296.0f));
}

// ln u for 0 < u < 1 (normal): u = m 2^e, m in (sqrt(1/2), sqrt 2]; ln m = 2z(1 + w/3 + ... + w^11/23)
__device__ __forceinline__ double dlog(double u)
{
    uint64_t bits = (uint64_t)__double_as_longlong(u);
    int e = (int)((bits >> 52) & 0x7ff) - 1023;
    bits = (bits & 0x000fffffffffffffULL) | 0x3ff0000000000000ULL;
    double m = __longlong_as_double((long long)bits);
    if (m > 0x1.6a09e667f3bcdp+0) { m = __dmul_rn(m, 0.5); e = e + 1; }
    const double z = __ddiv_rn(__dsub_rn(m, 1.0), __dadd_rn(m, 1.0));
    const double w = __dmul_rn(z, z);
    double s = 0x1.642c8590b2164p-5;
    s = __dadd_rn(__dmul_rn(s, w), 0x1.8618618618618p-5);
    s = __dadd_rn(__dmul_rn(s, w), 0x1.af286bca1af28p-5);
    s = __dadd_rn(__dmul_rn(s, w), 0x1.e1e1e1e1e1e1ep-5);
    s = __dadd_rn(__dmul_rn(s, w), 0x1.1111111111111p-4);
    s = __dadd_rn(__dmul_rn(s, w), 0x1.3b13b13b13b14p-4);
    s = __dadd_rn(__dmul_rn(s, w), 0x1.745d1745d1746p-4);
    s = __dadd_rn(__dmul_rn(s, w), 0x1.c71c71c71c71cp-4);
    s = __dadd_rn(__dmul_rn(s, w), 0x1.2492492492492p-3);
    s = __dadd_rn(__dmul_rn(s, w), 0x1.999999999999ap-3);
    s = __dadd_rn(__dmul_rn(s, w), 0x1.5555555555555p-2);
    s = __dadd_rn(__dmul_rn(s, w), 1.0);
    const double lnm = __dmul_rn(__dmul_rn(2.0, z), s);
    const double le = __dmul_rn((double)e, 0x1.62e42fefa39efp-1);
    return __dadd_rn(le, lnm);
}

// cos(2 pi u), sin(2 pi u), 0 <= u < 1: nearest quadrant, Taylor to x^18 / x^17 on [-pi/4, pi/4]
__device__ __forceinline__ void dsincos2pi(double u, double *c_out, double *s_out)
{
    const int kk = __double2int_rz(__dadd_rn(__dmul_rn(u, 4.0), 0.5));
    const double r = __dsub_rn(u, __dmul_rn((double)kk, 0.25));
    const double x = __dmul_rn(0x1.921fb54442d18p+2, r);
    const double x2 = __dmul_rn(x, x);
    double ps = 0x1.952c77030ad4ap-49;
    ps = __dadd_rn(__dmul_rn(ps, x2), -0x1.ae7f3e733b81fp-41);
    ps = __dadd_rn(__dmul_rn(ps, x2), 0x1.6124613a86d09p-33);
    ps = __dadd_rn(__dmul_rn(ps, x2), -0x1.ae64567f544e4p-26);
    ps = __dadd_rn(__dmul_rn(ps, x2), 0x1.71de3a556c734p-19);
    ps = __dadd_rn(__dmul_rn(ps, x2), -0x1.a01a01a01a01ap-13);
    ps = __dadd_rn(__dmul_rn(ps, x2), 0x1.1111111111111p-7);
    ps = __dadd_rn(__dmul_rn(ps, x2), -0x1.5555555555555p-3);
    ps = __dadd_rn(__dmul_rn(ps, x2), 1.0);
    const double sn = __dmul_rn(x, ps);
    double pc = -0x1.6827863b97d97p-53;
    pc = __dadd_rn(__dmul_rn(pc, x2), 0x1.ae7f3e733b81fp-45);
    pc = __dadd_rn(__dmul_rn(pc, x2), -0x1.93974a8c07c9dp-37);
    pc = __dadd_rn(__dmul_rn(pc, x2), 0x1.1eed8eff8d898p-29);
    pc = __dadd_rn(__dmul_rn(pc, x2), -0x1.27e4fb7789f5cp-22);
    pc = __dadd_rn(__dmul_rn(pc, x2), 0x1.a01a01a01a01ap-16);
    pc = __dadd_rn(__dmul_rn(pc, x2), -0x1.6c16c16c16c17p-10);
    pc = __dadd_rn(__dmul_rn(pc, x2), 0x1.5555555555555p-5);
    pc = __dadd_rn(__dmul_rn(pc, x2), -0x1.0000000000000p-1);
    pc = __dadd_rn(__dmul_rn(pc, x2), 1.0);
    const double cs = pc;
    switch (kk & 3) {
    case 0: *c_out = cs; *s_out = sn; break;
    case 1: *c_out = -sn; *s_out = cs; break;
    case 2: *c_out = -cs; *s_out = -sn; break;
    default: *c_out = sn; *s_out = -cs; break;
    }
}

// ----------------------------------------------------------------------- bit-sliced adders
// acc (NA planes, plane 0 = weight 1) += x (NB planes); no overflow check (caller sizes NA).
template <int NA, int NB>
__device__ __forceinline__ void bs_add(uint32_t (&acc)[NA], const uint32_t (&x)[NB])
{
    uint32_t carry = 0;
#pragma unroll
    for (int k = 0; k < NA; ++k) {
        if (k < NB) {
            const uint32_t a = acc[k];
            acc[k] = xor3(a, x[k], carry);
            carry = maj3(a, x[k], carry);
        } else {
            const uint32_t a = acc[k];
            acc[k] = a ^ carry;
            carry = a & carry;
        }
    }
}

// 32x32 bit-matrix transpose across a warp: before, lane j holds row j; after, lane i holds
// column i (bit j of the result = bit i of lane j's input).  All 32 lanes must participate.
__device__ __forceinline__ uint32_t transpose32(uint32_t x, int lane)
{
    // stage j: exchange j x j bit blocks with lane ^ j.  A lane with bit j clear keeps its low blocks (mask m) and takes
    // the partner's low blocks shifted up by j; a lane with bit j set keeps its high blocks (m << j) and takes the
    // partner's high blocks shifted down by j.  Both shifts are ONE rotation (left by j, or by 32 - j) because the bits
    // that wrap around land under the keep mask: per stage a shuffle, a funnel shift and a LOP3 select.
    uint32_t m = 0x0000FFFFu;
#pragma unroll
    for (int j = 16; j >= 1; j >>= 1) {
        const uint32_t y = __shfl_xor_sync(0xffffffffu, x, j);
        const bool up = (lane & j) != 0;
        const uint32_t keep = up ? (m << j) : m;
        const uint32_t rot = __funnelshift_l(y, y, up ? 32 - j : j);
        x = lop3<0xCA>(keep, x, rot);               // keep ? x : rot
        m ^= (m << (j >> 1));      // 0000FFFF -> 00FF00FF -> 0F0F0F0F -> 33333333 -> 55555555
    }
    return x;
}

// Sum over the 32 lanes of the warp of a bit-sliced count: after the call, lane l holds the
// integer total of spin-lane l:  sum_threads sum_k 2^k bit_l(acc[k]).
template <int P>
__device__ __forceinline__ uint32_t bs_warp_total(const uint32_t (&acc)[P], int n_planes, int lane)
{
    uint32_t total = 0;
#pragma unroll
    for (int k = 0; k < P; ++k) {
        if (k < n_planes) total += (uint32_t)__popc(transpose32(acc[k], lane)) << k;
    }
    return total;
}

}  // namespace sg
