// sg_pmj.cu — bit-packed (+-J) kernels, generic global-memory versions: any even L, any ladder.
//
// Layout: 32 disorder samples per uint32 (bit l = sample 32 w + l).
//   spins  [W][R][NT][2][H]   colour-compacted: entry n of colour c is site i with i>>1 == n,
//                             (x+y+z)&1 == c; bit 1 <-> S = +1
//   J      [W][2][3][H]       J[w][c][d][n] = bond (i -> i+e_d) owned by the site (c, n); bit 1 <-> J = -1
// In this layout the +-y, +-z neighbours of (c, row, m) sit at the same m in the neighbouring row
// of the other colour; one x-neighbour sits at the same (row, m), the other at m-1 or m+1
// depending on the row parity p = (c+y+z)&1.
#include "sg_device.cuh"
#include "sg_internal.h"

namespace sg {

// neighbour compact indices (all in the other colour's array) of the site (colour, n)
struct Nbr {
    int xp, xm, yp, ym, zp, zm;
};

__device__ __forceinline__ Nbr neighbours(const Dims &d, int colour, int n)
{
    const int row = n / d.Lh;
    const int m = n - row * d.Lh;
    const int z = row / d.L;
    const int y = row - z * d.L;
    const int p = (colour + y + z) & 1;
    const int side = row * d.Lh + (p ? (m + 1 == d.Lh ? 0 : m + 1) : (m == 0 ? d.Lh - 1 : m - 1));
    Nbr r;
    r.xp = p ? side : n;
    r.xm = p ? n : side;
    const int yp = (y + 1 == d.L) ? 0 : y + 1, ym = (y == 0) ? d.L - 1 : y - 1;
    const int zp = (z + 1 == d.L) ? 0 : z + 1, zm = (z == 0) ? d.L - 1 : z - 1;
    r.yp = (z * d.L + yp) * d.Lh + m;
    r.ym = (z * d.L + ym) * d.Lh + m;
    r.zp = (zp * d.L + y) * d.Lh + m;
    r.zm = (zm * d.L + y) * d.Lh + m;
    return r;
}

// canonical site i -> (colour, n)
__device__ __forceinline__ void site_to_compact(const Dims &d, int i, int &colour, int &n)
{
    const int x = i % d.L;
    const int yz = i / d.L;
    const int y = yz % d.L, z = yz / d.L;
    colour = (x + y + z) & 1;
    n = i >> 1;
}

// unsatisfied-bond words of the site (colour, n): u = s ^ s_nbr ^ j  (bit 1 <-> J S_i S_j = -1)
__device__ __forceinline__ void unsat_words(const Dims &d, int colour, int n, uint32_t s,
                                            const uint32_t *__restrict__ oth,
                                            const uint32_t *__restrict__ Jown,
                                            const uint32_t *__restrict__ Joth, uint32_t (&u)[6])
{
    const Nbr nb = neighbours(d, colour, n);
    const int H = d.H;
    u[0] = xor3(s, oth[nb.xp], Jown[n]);
    u[1] = xor3(s, oth[nb.xm], Joth[nb.xm]);
    u[2] = xor3(s, oth[nb.yp], Jown[H + n]);
    u[3] = xor3(s, oth[nb.ym], Joth[H + nb.ym]);
    u[4] = xor3(s, oth[nb.zp], Jown[2 * H + n]);
    u[5] = xor3(s, oth[nb.zm], Joth[2 * H + nb.zm]);
}

// 6 one-bit words -> 3-plane count (n0 + 2 n1 + 4 n2), 8 LOP3
__device__ __forceinline__ void count6(const uint32_t (&u)[6], uint32_t &n0, uint32_t &n1, uint32_t &n2)
{
    const uint32_t s0 = xor3(u[0], u[1], u[2]), c0 = maj3(u[0], u[1], u[2]);
    const uint32_t s1 = xor3(u[3], u[4], u[5]), c1 = maj3(u[3], u[4], u[5]);
    n0 = s0 ^ s1;
    const uint32_t k = s0 & s1;
    n1 = xor3(c0, c1, k);
    n2 = maj3(c0, c1, k);
}

// mask word = all ones iff r < thr, from c64 = (uint64)(0 - thr)  (thr in [0, 2^32])
__device__ __forceinline__ uint32_t lt_mask(uint32_t r, uint2 c64)
{
    const uint64_t v = (uint64_t)r + (((uint64_t)c64.y << 32) | c64.x);
    return (uint32_t)(v >> 32);
}

// Metropolis accept word, comparator path (|h| <= 1, monotone table):
// code c = (n2 n1 n0 ~a) accepted iff c >= k, k = #{c' in 0..6 : r >= thr[c']}.
__device__ __forceinline__ uint32_t accept_fast(uint32_t r, const uint2 (&c64)[7], uint32_t n0,
                                                uint32_t n1, uint32_t n2, uint32_t na)
{
    const uint32_t B0 = lt_mask(r, c64[0]), B1 = lt_mask(r, c64[1]), B2 = lt_mask(r, c64[2]);
    const uint32_t B3 = lt_mask(r, c64[3]), B4 = lt_mask(r, c64[4]), B5 = lt_mask(r, c64[5]);
    const uint32_t B6 = lt_mask(r, c64[6]);
    const uint32_t nK0 = xor3(xor3(B0, B1, B2), xor3(B3, B4, B5), B6);   // ~K0 (k even)
    const uint32_t K1 = lop3<LUT_K1>(B1, B3, B5);
    const uint32_t K2 = ~B3;
    const uint32_t g0 = na | nK0;
    const uint32_t g1 = lop3<LUT_GE>(n0, K1, g0);
    const uint32_t g2 = lop3<LUT_GE>(n1, K2, g1);
    return n2 | g2;
}

// general path (any h): select among the 14 class masks
__device__ __forceinline__ uint32_t accept_general(uint32_t r, const SlotTab &tb, uint32_t n0,
                                                   uint32_t n1, uint32_t n2, uint32_t a)
{
    uint32_t acc = 0;
#pragma unroll
    for (int nu = 0; nu < 7; ++nu) {
        const uint32_t e = ((nu & 1) ? n0 : ~n0) & ((nu & 2) ? n1 : ~n1) & ((nu & 4) ? n2 : ~n2);
        const uint32_t b0 = lt_mask(r, tb.c64g[nu][0]), b1 = lt_mask(r, tb.c64g[nu][1]);
        acc |= e & ((a & b1) | (~a & b0));
    }
    return acc;
}

// ------------------------------------------------------------------------------------ init
__global__ void k_init_J_pmj(Dims d, uint32_t *__restrict__ J)
{
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= (long long)d.W * d.N) return;
    const int i = (int)(tid % d.N);
    const int w = (int)(tid / d.N);
    int c, n;
    site_to_compact(d, i, c, n);
    const uint4 o = philox4x32_10((uint32_t)i, 0u, (uint32_t)(w + (d.s_first >> 5)), ctr3(1, 0, 0), d.k0, d.k1);
    uint32_t *base = J + ((size_t)(w * 2 + c) * 3) * d.H + n;
    base[0] = o.x;
    base[d.H] = o.y;
    base[2 * d.H] = o.z;
}

__global__ void k_init_S_pmj(Dims d, uint32_t *__restrict__ spins)
{
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = (long long)d.W * d.R * d.NT * d.N;
    if (tid >= total) return;
    const int i = (int)(tid % d.N);
    const int sys = (int)(tid / d.N);
    const int t = sys % d.NT, a = (sys / d.NT) % d.R, w = sys / (d.NT * d.R);
    int c, n;
    site_to_compact(d, i, c, n);
    const uint4 o = philox4x32_10((uint32_t)i, 0u, (uint32_t)(w + (d.s_first >> 5)), ctr3(2, a, t), d.k0, d.k1);
    spins[((size_t)sys * 2 + c) * d.H + n] = o.x;
}

// ----------------------------------------------------------------------------------- sweep
// One thread per (system, quad of 4 consecutive same-colour sites) = one Philox call (R6).
__global__ void __launch_bounds__(256)
k_sweep_pmj(Dims d, uint32_t *__restrict__ spins, const uint32_t *__restrict__ J,
            const SlotTab *__restrict__ tab, uint32_t sweep, int colour)
{
    const int Q = d.H >> 2;
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= (long long)d.W * d.R * d.NT * Q) return;
    const int q = (int)(tid % Q);
    const int sys = (int)(tid / Q);
    const int t = sys % d.NT, a = (sys / d.NT) % d.R, w = sys / (d.NT * d.R);
    uint32_t *act = spins + ((size_t)sys * 2 + colour) * d.H;
    const uint32_t *oth = spins + ((size_t)sys * 2 + (1 - colour)) * d.H;
    const uint32_t *Jown = J + ((size_t)(w * 2 + colour) * 3) * d.H;
    const uint32_t *Joth = J + ((size_t)(w * 2 + 1 - colour) * 3) * d.H;

    uint4 s4 = *reinterpret_cast<uint4 *>(act + 4 * q);
    const uint4 r4 = philox4x32_10((uint32_t)q, 2u * sweep + (uint32_t)colour, (uint32_t)(w + (d.s_first >> 5)), ctr3(3, a, t), d.k0, d.k1);
    uint32_t s[4] = {s4.x, s4.y, s4.z, s4.w};
    const uint32_t r[4] = {r4.x, r4.y, r4.z, r4.w};
    const SlotTab &tb = tab[t];
    uint2 c64[7];
#pragma unroll
    for (int c = 0; c < 7; ++c) c64[c] = tb.c64[c];
    const uint32_t amask = d.neg_h ? 0xffffffffu : 0u;      // a = s ^ amask
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        uint32_t u[6], n0, n1, n2;
        unsat_words(d, colour, 4 * q + e, s[e], oth, Jown, Joth, u);
        count6(u, n0, n1, n2);
        const uint32_t av = s[e] ^ amask;
        const uint32_t acc = d.fast_accept ? accept_fast(r[e], c64, n0, n1, n2, ~av)
                                           : accept_general(r[e], tb, n0, n1, n2, av);
        s[e] ^= acc;
    }
    *reinterpret_cast<uint4 *>(act + 4 * q) = make_uint4(s[0], s[1], s[2], s[3]);
}

// ---------------------------------------------------------------------------------- energy
// One warp per system: per-lane U = number of unsatisfied bonds (sum over colour-0 sites of their
// 6 bonds covers every bond once), M = sum of spins.  Bit-sliced accumulation, then a warp
// transpose + popc per plane.
__global__ void __launch_bounds__(128)
k_energy_pmj(Dims d, const uint32_t *__restrict__ spins, const uint32_t *__restrict__ J,
             int64_t *__restrict__ U, int32_t *__restrict__ M)
{
    const int lane = threadIdx.x & 31;
    const int sys = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (sys >= d.W * d.R * d.NT) return;
    const int t = sys % d.NT, a = (sys / d.NT) % d.R, w = sys / (d.NT * d.R);
    const uint32_t *s0 = spins + ((size_t)sys * 2) * d.H;
    const uint32_t *s1 = s0 + d.H;
    const uint32_t *J0 = J + ((size_t)(w * 2) * 3) * d.H;
    const uint32_t *J1 = J + ((size_t)(w * 2 + 1) * 3) * d.H;

    uint32_t bigU[16], bigM[16], inU[7], inM[6];
#pragma unroll
    for (int k = 0; k < 16; ++k) bigU[k] = bigM[k] = 0;
#pragma unroll
    for (int k = 0; k < 7; ++k) inU[k] = 0;
#pragma unroll
    for (int k = 0; k < 6; ++k) inM[k] = 0;
    int pending = 0;
    for (int n = lane; n < d.H; n += 32) {
        const uint32_t sa = s0[n], sb = s1[n];
        uint32_t u[6], x[3];
        unsat_words(d, 0, n, sa, s1, J0, J1, u);
        count6(u, x[0], x[1], x[2]);
        bs_add(inU, x);
        const uint32_t mm[2] = {sa ^ sb, sa & sb};
        bs_add(inM, mm);
        if (++pending == 16) {
            bs_add(bigU, inU);
            bs_add(bigM, inM);
#pragma unroll
            for (int k = 0; k < 7; ++k) inU[k] = 0;
#pragma unroll
            for (int k = 0; k < 6; ++k) inM[k] = 0;
            pending = 0;
        }
    }
    bs_add(bigU, inU);
    bs_add(bigM, inM);
    const int per_thread = (d.H + 31) / 32;
    int pu = 1, pm = 1;
    while ((1 << pu) <= 6 * per_thread) ++pu;
    while ((1 << pm) <= 2 * per_thread) ++pm;
    const uint32_t totU = bs_warp_total(bigU, pu, lane);
    const uint32_t totM = bs_warp_total(bigM, pm, lane);
    const size_t o = ((size_t)(w * 32 + lane) * d.R + a) * d.NT + t;
    U[o] = (int64_t)totU;
    M[o] = 2 * (int32_t)totM - d.N;
}

// -------------------------------------------------------------------------------------- PT
// One warp per (word, replica, pair): lane l decides for sample 32 w + l (R12).
__global__ void __launch_bounds__(128)
k_pt_decide_pmj(Dims d, const int64_t *__restrict__ U, const int32_t *__restrict__ M,
                const SlotTab *__restrict__ tab, const double *__restrict__ exp_tab, double h,
                uint32_t exchange, int npairs, uint32_t *__restrict__ swapmask,
                unsigned long long *__restrict__ pt_acc)
{
    const int lane = threadIdx.x & 31;
    const int g = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (g >= d.W * d.R * npairs) return;
    const int pair = g % npairs, a = (g / npairs) % d.R, w = g / (npairs * d.R);
    const int t = (int)(exchange & 1u) + 2 * pair;
    const int s = w * 32 + lane;
    const size_t o = ((size_t)s * d.R + a) * d.NT + t;
    const double Et = __dsub_rn((double)(2 * U[o] - 3 * (int64_t)d.N), __dmul_rn(h, (double)M[o]));
    const double Eu = __dsub_rn((double)(2 * U[o + 1] - 3 * (int64_t)d.N), __dmul_rn(h, (double)M[o + 1]));
    const double x = __dmul_rn(__dsub_rn(tab[t].beta, tab[t + 1].beta), __dsub_rn(Et, Eu));
    const uint4 r = philox4x32_10(0u, exchange, (uint32_t)(s + d.s_first), ctr3(4, a, t), d.k0, d.k1);
    const bool accept = (x >= 0.0) || ((uint64_t)r.x < dexp64(exp_tab, -x));
    const uint32_t mask = __ballot_sync(0xffffffffu, accept && s < d.n_samples);
    if (lane == 0) {
        swapmask[(size_t)(w * d.R + a) * (d.NT / 2) + pair] = mask;
        if (mask) atomicAdd(&pt_acc[t], (unsigned long long)__popc(mask));
    }
}

// One CTA per (word, replica, pair) - the word index is gridDim.x (limit 2^31 - 1; y and z stop at 65535): reads the pair's mask once and leaves if no lane swaps (the common
// case on a wide ladder); otherwise trades the selected lanes of the two configurations and of their U, M.
__global__ void __launch_bounds__(256)
k_pt_swap_pmj(Dims d, uint32_t *__restrict__ spins, const uint32_t *__restrict__ swapmask,
              uint32_t exchange, int npairs, int64_t *__restrict__ U, int32_t *__restrict__ M)
{
    const int w = blockIdx.x, a = blockIdx.y, pair = blockIdx.z;
    const uint32_t mask = swapmask[(size_t)(w * d.R + a) * (d.NT / 2) + pair];
    if (mask == 0) return;
    const int t = (int)(exchange & 1u) + 2 * pair;
    const size_t sys = ((size_t)w * d.R + a) * d.NT + t;
    uint4 *A = reinterpret_cast<uint4 *>(spins + sys * d.N);
    uint4 *B = reinterpret_cast<uint4 *>(spins + (sys + 1) * d.N);
    for (int j = threadIdx.x; j < (d.N >> 2); j += blockDim.x) {
        uint4 x = A[j], y = B[j];
        uint32_t dd;
        dd = (x.x ^ y.x) & mask; x.x ^= dd; y.x ^= dd;
        dd = (x.y ^ y.y) & mask; x.y ^= dd; y.y ^= dd;
        dd = (x.z ^ y.z) & mask; x.z ^= dd; y.z ^= dd;
        dd = (x.w ^ y.w) & mask; x.w ^= dd; y.w ^= dd;
        A[j] = x;
        B[j] = y;
    }
    if (threadIdx.x < 32 && ((mask >> threadIdx.x) & 1u)) {
        const size_t o = ((size_t)(w * 32 + threadIdx.x) * d.R + a) * d.NT + t;
        const int64_t u = U[o]; U[o] = U[o + 1]; U[o + 1] = u;
        const int32_t m = M[o]; M[o] = M[o + 1]; M[o + 1] = m;
    }
}

// ------------------------------------------------------------------------------------ hash
// One warp per system: sum over its words of mix64(index, word) (order-free; sg_get_state_hash).
__device__ __forceinline__ uint64_t mix64(uint64_t x)
{
    x ^= x >> 30; x *= 0xbf58476d1ce4e5b9ULL;
    x ^= x >> 27; x *= 0x94d049bb133111ebULL;
    x ^= x >> 31;
    return x;
}

__global__ void __launch_bounds__(128)
k_hash_words(const uint32_t *__restrict__ words, long long n_sys, int words_per_sys, uint64_t *__restrict__ out)
{
    const int lane = threadIdx.x & 31;
    const long long sys = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (sys >= n_sys) return;
    const uint32_t *p = words + (size_t)sys * words_per_sys;
    uint64_t h = 0;
    for (int i = lane; i < words_per_sys; i += 32) h += mix64(((uint64_t)(uint32_t)i << 32) | p[i]);
    for (int o = 16; o; o >>= 1) h += __shfl_xor_sync(0xffffffffu, h, o);
    if (lane == 0) out[sys] = h;
}

// ------------------------------------------------------------------------------- measurement
// Plane histograms of the differing-site indicator d_j = [S^a_j != S^b_j] (S^a S^b = 1 - 2 d):
// hist[h][m] = #{j : d_j = 1, coordinate_h(j) = m}, h = x, y, z, x+y, x-y, x+z, x-z, y+z, y-z (mod L).
// They are sufficient statistics for q(0) and the 12 wave vectors of R8.
// v1: one warp per (word, slot, pair), lane l counts for sample 32 w + l in shared memory.
__global__ void __launch_bounds__(32)
k_hist_pmj(Dims d, const uint32_t *__restrict__ spins, int w0, uint16_t *__restrict__ hist)
{
    extern __shared__ uint16_t sh[];            // [N_HIST][L][32]
    const int lane = threadIdx.x;
    const int L = d.L;
    int g = blockIdx.x;                          // ((w - w0) * NT + t) * P + pair
    const int pair = g % d.P;  g /= d.P;
    const int t = g % d.NT;    g /= d.NT;
    const int w = w0 + g;
    int ra = 0, rb = 1;
    {   // pair index -> (a, b), a < b, lexicographic
        int p = 0;
        for (int a = 0; a < d.R; ++a)
            for (int b = a + 1; b < d.R; ++b) {
                if (p == pair) { ra = a; rb = b; }
                ++p;
            }
    }
    const uint32_t *A = spins + ((((size_t)w * d.R + ra) * d.NT + t) * 2) * d.H;
    const uint32_t *B = spins + ((((size_t)w * d.R + rb) * d.NT + t) * 2) * d.H;
    for (int k = 0; k < N_HIST * L; ++k) sh[k * 32 + lane] = 0;
    for (int z = 0; z < L; ++z)
        for (int y = 0; y < L; ++y) {
            const int row = z * L + y;
            int rowcnt = 0;
            for (int c = 0; c < 2; ++c) {
                const int p = (c + y + z) & 1;
                for (int m = 0; m < d.Lh; ++m) {
                    const int idx = c * d.H + row * d.Lh + m;
                    const int bit = (int)(((A[idx] ^ B[idx]) >> lane) & 1u);
                    const int x = 2 * m + p;
                    rowcnt += bit;
                    int b;
                    sh[(0 * L + x) * 32 + lane] += bit;
                    b = x + y;      if (b >= L) b -= L;  sh[(3 * L + b) * 32 + lane] += bit;
                    b = x - y;      if (b < 0) b += L;   sh[(4 * L + b) * 32 + lane] += bit;
                    b = x + z;      if (b >= L) b -= L;  sh[(5 * L + b) * 32 + lane] += bit;
                    b = x - z;      if (b < 0) b += L;   sh[(6 * L + b) * 32 + lane] += bit;
                }
            }
            int b;
            sh[(1 * L + y) * 32 + lane] += rowcnt;
            sh[(2 * L + z) * 32 + lane] += rowcnt;
            b = y + z;  if (b >= L) b -= L;  sh[(7 * L + b) * 32 + lane] += rowcnt;
            b = y - z;  if (b < 0) b += L;   sh[(8 * L + b) * 32 + lane] += rowcnt;
        }
    const size_t s_local = (size_t)(w - w0) * 32 + lane;
    uint16_t *out = hist + ((s_local * d.NT + t) * d.P + pair) * (size_t)(N_HIST * L);
    for (int k = 0; k < N_HIST * L; ++k) out[k] = sh[k * 32 + lane];
}

// -------------------------------------------------------------------- pack / unpack / getters
// canonical bytes [ns][R][NT][N] (+-1) <-> packed words, samples [s0, s0+ns)
__global__ void k_unpack_pmj(Dims d, const uint32_t *__restrict__ spins, int s0, int ns, int8_t *__restrict__ out)
{
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = (long long)ns * d.R * d.NT * d.N;
    if (tid >= total) return;
    const int i = (int)(tid % d.N);
    long long g = tid / d.N;
    const int t = (int)(g % d.NT);  g /= d.NT;
    const int a = (int)(g % d.R);   g /= d.R;
    const int s = s0 + (int)g;
    int c, n;
    site_to_compact(d, i, c, n);
    const size_t sys = ((size_t)(s >> 5) * d.R + a) * d.NT + t;
    const uint32_t wv = spins[(sys * 2 + c) * d.H + n];
    out[tid] = ((wv >> (s & 31)) & 1u) ? 1 : -1;
}

// one thread per (word-site of the touched words): merges the lanes of samples [s0, s0+ns)
__global__ void k_pack_pmj(Dims d, uint32_t *__restrict__ spins, int s0, int ns, const int8_t *__restrict__ in)
{
    const int w_first = s0 >> 5, w_last = (s0 + ns - 1) >> 5;
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = (long long)(w_last - w_first + 1) * d.R * d.NT * d.N;
    if (tid >= total) return;
    const int i = (int)(tid % d.N);
    long long g = tid / d.N;
    const int t = (int)(g % d.NT);  g /= d.NT;
    const int a = (int)(g % d.R);   g /= d.R;
    const int w = w_first + (int)g;
    int c, n;
    site_to_compact(d, i, c, n);
    const size_t sys = ((size_t)w * d.R + a) * d.NT + t;
    uint32_t wv = spins[(sys * 2 + c) * d.H + n];
    for (int l = 0; l < 32; ++l) {
        const int s = w * 32 + l;
        if (s < s0 || s >= s0 + ns) continue;
        const int8_t v = in[(((size_t)(s - s0) * d.R + a) * d.NT + t) * d.N + i];
        wv = (wv & ~(1u << l)) | ((v > 0 ? 1u : 0u) << l);
    }
    spins[(sys * 2 + c) * d.H + n] = wv;
}

__global__ void k_couplings_pmj(Dims d, const uint32_t *__restrict__ J, int s0, int ns, float *__restrict__ out)
{
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = (long long)ns * 3 * d.N;
    if (tid >= total) return;
    const int i = (int)(tid % d.N);
    const int dd = (int)((tid / d.N) % 3);
    const int s = s0 + (int)(tid / (3LL * d.N));
    int c, n;
    site_to_compact(d, i, c, n);
    const uint32_t wv = J[((size_t)((s >> 5) * 2 + c) * 3 + dd) * d.H + n];
    out[tid] = ((wv >> (s & 31)) & 1u) ? -1.0f : 1.0f;
}

// --------------------------------------------------------------------------------- launchers
static inline unsigned blocks_for(long long n, int per) { return (unsigned)((n + per - 1) / per); }

int launch_init_pmj(sg_ctx *c)
{
    const Dims &d = c->d;
    k_init_J_pmj<<<blocks_for((long long)d.W * d.N, 256), 256, 0, c->stream>>>(d, c->J);
    k_init_S_pmj<<<blocks_for((long long)d.W * d.R * d.NT * d.N, 256), 256, 0, c->stream>>>(d, c->spins);
    return 2;
}

int launch_sweep_pmj(sg_ctx *c, uint64_t sweep)
{
    const Dims &d = c->d;
    const long long n = (long long)d.W * d.R * d.NT * (d.H >> 2);
    for (int colour = 0; colour < 2; ++colour)
        k_sweep_pmj<<<blocks_for(n, 256), 256, 0, c->stream>>>(d, c->spins, c->J, c->tab, (uint32_t)sweep, colour);
    return 2;
}

int launch_energy_pmj(sg_ctx *c)
{
    const Dims &d = c->d;
    k_energy_pmj<<<blocks_for((long long)d.W * d.R * d.NT, 4), 128, 0, c->stream>>>(d, c->spins, c->J, c->U, c->M);
    return 1;
}

int launch_pt_pmj(sg_ctx *c, uint64_t exchange)
{
    const Dims &d = c->d;
    const int npairs = (d.NT - (int)(exchange & 1)) / 2;
    if (npairs <= 0) return 0;
    k_pt_decide_pmj<<<blocks_for((long long)d.W * d.R * npairs, 4), 128, 0, c->stream>>>(
        d, c->U, c->M, c->tab, c->exp64_tab, c->h, (uint32_t)exchange, npairs, c->swapmask, c->pt_acc);
    k_pt_swap_pmj<<<dim3(d.W, d.R, npairs), 256, 0, c->stream>>>(d, c->spins, c->swapmask, (uint32_t)exchange, npairs,
                                                                 c->U, c->M);
    return 2;
}

int launch_hash(sg_ctx *c, uint64_t *dev_out)
{
    const Dims &d = c->d;
    const long long n_sys = (long long)d.W * d.R * d.NT;
    const int wps = is_packed(c) ? d.N : d.N / 4;
    const uint32_t *words = is_packed(c) ? c->spins : reinterpret_cast<const uint32_t *>(c->spins8);
    k_hash_words<<<blocks_for(n_sys, 4), 128, 0, c->stream>>>(words, n_sys, wps, dev_out);
    return 1;
}

int launch_hist_pmj(sg_ctx *c, int s0, int ns)
{
    const Dims &d = c->d;
    const int w0 = s0 >> 5, nw = (ns + 31) >> 5;
    const size_t sh = (size_t)N_HIST * d.L * 32 * sizeof(uint16_t);
    k_hist_pmj<<<(unsigned)(nw * d.NT * d.P), 32, sh, c->stream>>>(d, c->spins, w0, c->hist);
    return 1;
}

int launch_unpack_pmj(sg_ctx *c, int s0, int ns)
{
    const Dims &d = c->d;
    k_unpack_pmj<<<blocks_for((long long)ns * d.R * d.NT * d.N, 256), 256, 0, c->stream>>>(d, c->spins, s0, ns, c->stage8);
    return 1;
}

int launch_pack_pmj(sg_ctx *c, int s0, int ns)
{
    const Dims &d = c->d;
    const int nw = ((s0 + ns - 1) >> 5) - (s0 >> 5) + 1;
    k_pack_pmj<<<blocks_for((long long)nw * d.R * d.NT * d.N, 256), 256, 0, c->stream>>>(d, c->spins, s0, ns, c->stage8);
    return 1;
}

int launch_couplings_pmj(sg_ctx *c, int s0, int ns, float *dev_out)
{
    const Dims &d = c->d;
    k_couplings_pmj<<<blocks_for((long long)ns * 3 * d.N, 256), 256, 0, c->stream>>>(d, c->J, s0, ns, dev_out);
    return 1;
}

}  // namespace sg
