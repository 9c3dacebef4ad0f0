// sg_ladder.cu — the fast +-J path for lattices whose temperature ladder fits in shared memory (L = 4 .. 16).
//
// One CTA owns one (packed word w, replica a) ladder: its NT systems (NT * N words) and the word's couplings (3 N words)
// stay in shared memory for `n_sweeps` consecutive checkerboard sweeps and the exchanges between them, so global memory is
// touched once per launch.  A ladder larger than one SM is split over a cluster of two CTAs (half of the slots each).
// The unit of work is a quad: 4 consecutive same-colour sites = one Philox call (R6); its 24 coupling words live in
// registers across the systems handled with it.  Three shared-memory layouts, by the row length L/2 in words:
//   * whole quads per row (L = 8, 16): canonical order; thread = (quad, group of slots); 128-bit neighbour accesses;
//   * even, not whole quads (L = 4, 12): "pair" layout [low 64-bit pairs][high pairs]; items (block of 32 quads, slot)
//     dealt out evenly over 12 warps; 64-bit neighbour accesses without bank conflicts;
//   * odd (L = 6, 10): "planar" layout, word e of every quad in array e; same items; 32-bit unit-stride accesses.
// Three instantiations per (L, compare variant), template parameter PTM: 0 = plain sweeps (no exchange code; the last,
// half-empty wave of ladders goes to two CTAs each), 1 = exchanges by a one-warp-per-slot recount (+ the cross pair of a
// split ladder through distributed shared memory), 2 = exchanges by the warp-per-pair colour-1 half sweep (energy counts in
// registers, decision and swap by the same warp).
// Bit-sliced arithmetic as in sg_pmj.cu: per word-site 6 XOR3 + 8 (count) + 4 (compare / flip) + 3 carries + 5 (Philox
// share) = 26 ALU-pipe lane-ops with the binary-search compare; the Philox products and the threshold selection are IMADs on
// the FMA pipe.
#include "sg_accept.cuh"
#include "sg_device.cuh"
#include "sg_internal.h"

#include <algorithm>
#include <type_traits>

namespace sg {

struct LadderArgs {
    Dims d;
    uint32_t *spins;          // state the launch starts from
    uint32_t *spins_out;      // where it leaves the state (the same buffer, or the second one: see sg_run)
    const uint32_t *J;
    const SlotTab *tab;
    uint32_t rk[20];          // Philox round keys: rk[2r] = k0 + r*0x9E3779B9, rk[2r+1] = k1 + r*0xBB67AE85
    uint32_t pad0;
    uint32_t sweep0;          // global index of the first sweep of this launch
    int n_sweeps;
    int G;                    // system groups: thread (q, g) handles systems g, g+G, ...
    int pt_every;             // > 0: exchanges fused in (after every pt_every-th sweep, global sweep index)
    uint64_t exchange0;       // global index of the first exchange of this launch
    const double *exp_tab;    // dexp64 table (R12)
    double h;
    uint32_t one, mone;       // run-time 1 and 0xFFFFFFFF (sg_accept.cuh)
    int64_t *U;               // the kernel's own energies after the last exchange of the launch (see sg_ladder8.cu)
    int32_t *M;
    unsigned long long *pt_acc;
    int use_tab;              // shared memory has room for the energy tables (neighbour indices + gathered couplings)
    int n_full;               // CTAs [0, n_full) own a whole ladder; launches without exchanges may split the last ladders
                              // of the grid into two CTAs each (half of the slots) so that the last wave fills the SMs
    int nt_res;               // slots resident in one CTA: NT, or ceil(NT / 2) when every ladder is split over two CTAs (`split`)
    int split;                // 1: every ladder is split (launches with exchanges: the two CTAs form a cluster and the slot pair
                              // across them exchanges through distributed shared memory)
    int use_spw;              // pair layout: room for the offset table of the system-per-warp exchange half sweep
};

__device__ __forceinline__ uint4 philox_rk(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                           const uint32_t (&rk)[20])
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

// all ones iff r < thr, c64 = (uint64)(0 - thr): high word of r + c64.  ptxas emits one IADD3 (carry
// out, ALU pipe) + one IMAD.X (c64.hi + carry, FMA pipe); a mad.wide formulation is split the same way.
__device__ __forceinline__ uint32_t lt_mask64(uint32_t r, uint2 c64)
{
    const uint64_t v = (uint64_t)r + (((uint64_t)c64.y << 32) | c64.x);
    return (uint32_t)(v >> 32);
}

// Metropolis update of one word-site: returns the new spin word.  u0..u5 are the unsatisfied-bond
// words, na = ~a (a = field alignment), B[c] = all ones iff r < thr[code c]  (comparator path).
__device__ __forceinline__ uint32_t flip_word(uint32_t s, uint32_t u0, uint32_t u1, uint32_t u2, uint32_t u3,
                                              uint32_t u4, uint32_t u5, uint32_t na, const uint32_t (&B)[7])
{
    const uint32_t s0 = xor3(u0, u1, u2), c0 = maj3(u0, u1, u2);
    const uint32_t s1 = xor3(u3, u4, u5), c1 = maj3(u3, u4, u5);
    const uint32_t n0 = s0 ^ s1;
    const uint32_t k = s0 & s1;
    const uint32_t n1 = xor3(c0, c1, k);
    const uint32_t n2 = maj3(c0, c1, k);
    const uint32_t nK0 = xor3(xor3(B[0], B[1], B[2]), xor3(B[3], B[4], B[5]), B[6]);
    const uint32_t K1 = lop3<LUT_K1>(B[1], B[3], B[5]);
    const uint32_t g0 = na | nK0;
    const uint32_t g1 = lop3<LUT_GE>(n0, K1, g0);
    const uint32_t g2 = lop3<(0xF0 & 0xCC) | ((0xF0 ^ 0xCC) & 0xAA)>(n1, B[3], g1);   // GE(n1, K2, g1) with K2 = ~B3 folded in
    return lop3<LUT_FLIP>(s, n2, g2);
}

template <int L>
struct Geo {
    static constexpr int Lh = L / 2, N = L * L * L, H = N / 2, Q = H / 4;
    static constexpr bool VEC = (Lh % 4) == 0;
    static constexpr int QR = VEC ? Lh / 4 : 1;     // quads per row (vector path)
    // Rows of an even number of words that are not whole quads (L = 4, 12): every colour block of H words is kept in
    // shared memory as two arrays of 64-bit pairs, [low pairs of the quads][high pairs of the quads].  A lane's quad is
    // then two unit-stride 64-bit accesses, and so is every +-y / +-z neighbour (they start at an even word, i.e. on a
    // pair, but not on a quad): no shared-memory bank conflicts, where 64-bit pairs at a 16-byte stride had 2-way ones.
    static constexpr bool PAIR = !VEC && (Lh % 2) == 0;
    // position of compact index n (< H) inside its colour block
    // Rows of an ODD number of words (L = 6, 10): nothing beyond the quad is aligned, every neighbour is a 32-bit access at
    // a 16-byte stride over the lanes (4-way bank conflicts).  Planar layout: a colour block is kept as four arrays, word e
    // of every quad; the lanes of a warp (consecutive quads, same e) then touch consecutive words for every neighbour.
    static constexpr bool PLANAR = !VEC && !PAIR;
    static __host__ __device__ constexpr int pos(int n)
    {
        return PAIR ? ((n >> 1) & 1) * (H / 2) + ((n >> 2) << 1) + (n & 1) : PLANAR ? (n & 3) * Q + (n >> 2) : n;
    }
    // (L = 8 has its own kernel, sg_ladder8.cu; this one runs it when that kernel's ladder does not fit: one CTA per SM)
    static constexpr int MAXT = VEC ? 512 : 384;
    static constexpr int MINB = 1;
};

// Per-lane U (unsatisfied bonds) and M (sum of spins) of one system resident in shared memory, by ONE warp:
// the six bonds of every colour-0 site cover each bond once; bit-sliced accumulation (flush every 16 sites),
// then one warp transpose + popc per plane.  Same arithmetic as k_energy_pmj (sg_pmj.cu), compile-time L.
template <int L>
__device__ __forceinline__ void ladder_energy(const uint32_t *__restrict__ Ssys, const uint32_t *__restrict__ Jsm, int lane,
                                              int &U, int &M)
{
    constexpr int Lh = L / 2, N = L * L * L, H = N / 2;
    const uint32_t *s0 = Ssys, *s1 = Ssys + H;
    const uint32_t *J0 = Jsm, *J1 = Jsm + 3 * H;
    uint32_t bigU[16], bigM[16], inU[7], inM[6];
#pragma unroll
    for (int k = 0; k < 16; ++k) bigU[k] = bigM[k] = 0;
#pragma unroll
    for (int k = 0; k < 7; ++k) inU[k] = 0;
#pragma unroll
    for (int k = 0; k < 6; ++k) inM[k] = 0;
    int pending = 0;
    for (int n = lane; n < H; n += 32) {
        const int row = n / Lh, m = n - row * Lh;
        const int z = row / L, y = row - z * L;
        const int p = (y + z) & 1;                                     // colour 0
        const int sd = row * Lh + (p ? (m + 1 == Lh ? 0 : m + 1) : (m == 0 ? Lh - 1 : m - 1));
        const int xp = p ? sd : n, xm = p ? n : sd;
        const int yp = (z * L + (y + 1 == L ? 0 : y + 1)) * Lh + m, ym = (z * L + (y == 0 ? L - 1 : y - 1)) * Lh + m;
        const int zp = ((z + 1 == L ? 0 : z + 1) * L + y) * Lh + m, zm = ((z == 0 ? L - 1 : z - 1) * L + y) * Lh + m;
        constexpr auto P = Geo<L>::pos;                               // shared-memory position of a compact index
        const uint32_t sa = s0[P(n)], sb = s1[P(n)];
        const uint32_t u0 = xor3(sa, s1[P(xp)], J0[P(n)]), u1 = xor3(sa, s1[P(xm)], J1[P(xm)]);
        const uint32_t u2 = xor3(sa, s1[P(yp)], J0[H + P(n)]), u3 = xor3(sa, s1[P(ym)], J1[H + P(ym)]);
        const uint32_t u4 = xor3(sa, s1[P(zp)], J0[2 * H + P(n)]), u5 = xor3(sa, s1[P(zm)], J1[2 * H + P(zm)]);
        const uint32_t a0 = xor3(u0, u1, u2), c0 = maj3(u0, u1, u2);
        const uint32_t a1 = xor3(u3, u4, u5), c1 = maj3(u3, u4, u5);
        const uint32_t kk = a0 & a1;
        const uint32_t x[3] = {a0 ^ a1, xor3(c0, c1, kk), maj3(c0, c1, kk)};
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
    constexpr int per_thread = (H + 31) / 32;
    int pu = 1, pm = 1;
    while ((1 << pu) <= 6 * per_thread) ++pu;
    while ((1 << pm) <= 2 * per_thread) ++pm;
    U = (int)bs_warp_total(bigU, pu, lane);
    M = 2 * (int)bs_warp_total(bigM, pm, lane) - N;
}

// The same recount with everything that does not depend on the system taken from two tables built once per launch:
// idxT[n] = the six neighbour indices of colour-0 site n (16 bits each), JgT[n] = its six coupling words in the same
// order (+x, -x, +y, -y, +z, -z); four sites per step, their counts summed by a small adder tree before they are
// added to the running bit-sliced totals.  ~2.3x fewer instructions per site than ladder_energy.
template <int L>
__device__ __forceinline__ void ladder_energy_tab(const uint32_t *__restrict__ Ssys, const uint4 *__restrict__ idxT,
                                                  const uint32_t *__restrict__ JgT, int lane, int &U, int &M)
{
    constexpr int N = L * L * L, H = N / 2;
    // per thread: at most ceil(H / 32) sites -> U <= 6 sites, spin count <= 2 sites: just enough planes
    constexpr int SPT = (H + 31) / 32;
    constexpr int PU = SPT * 6 < 8 ? 3 : SPT * 6 < 16 ? 4 : SPT * 6 < 32 ? 5 : SPT * 6 < 64 ? 6 : SPT * 6 < 128 ? 7 : SPT * 6 < 256 ? 8 : 9;
    constexpr int PM = SPT * 2 < 8 ? 3 : SPT * 2 < 16 ? 4 : SPT * 2 < 32 ? 5 : SPT * 2 < 64 ? 6 : SPT * 2 < 128 ? 7 : 8;
    static_assert(SPT * 6 < 512 && SPT * 2 < 256, "plane counts");
    const uint32_t *s0 = Ssys, *s1 = Ssys + H;
    uint32_t bigU[PU], bigM[PM];
#pragma unroll
    for (int k = 0; k < PU; ++k) bigU[k] = 0;
#pragma unroll
    for (int k = 0; k < PM; ++k) bigM[k] = 0;
    for (int n0 = lane; n0 < H; n0 += 128) {
        uint32_t w[4][3], sw[8];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const int n = n0 + 32 * e;
            if (n < H) {
                const uint4 ii = idxT[n];
                const uint2 j01 = *reinterpret_cast<const uint2 *>(JgT + 6 * n);
                const uint2 j23 = *reinterpret_cast<const uint2 *>(JgT + 6 * n + 2);
                const uint2 j45 = *reinterpret_cast<const uint2 *>(JgT + 6 * n + 4);
                const uint32_t sa = s0[ii.w];                         // ii.w = position of n in its colour block
                const uint32_t u0 = xor3(sa, s1[ii.x & 0xffffu], j01.x), u1 = xor3(sa, s1[ii.x >> 16], j01.y);
                const uint32_t u2 = xor3(sa, s1[ii.y & 0xffffu], j23.x), u3 = xor3(sa, s1[ii.y >> 16], j23.y);
                const uint32_t u4 = xor3(sa, s1[ii.z & 0xffffu], j45.x), u5 = xor3(sa, s1[ii.z >> 16], j45.y);
                const uint32_t a0 = xor3(u0, u1, u2), c0 = maj3(u0, u1, u2);
                const uint32_t a1 = xor3(u3, u4, u5), c1 = maj3(u3, u4, u5);
                const uint32_t kk = a0 & a1;
                w[e][0] = a0 ^ a1;
                w[e][1] = xor3(c0, c1, kk);
                w[e][2] = maj3(c0, c1, kk);
                sw[2 * e] = sa;
                sw[2 * e + 1] = s1[ii.w];
            } else {
                w[e][0] = w[e][1] = w[e][2] = 0u;
                sw[2 * e] = sw[2 * e + 1] = 0u;
            }
        }
        uint32_t ab[4], cd[4], U5[5];
        bs_sum<3>(w[0], w[1], ab);
        bs_sum<3>(w[2], w[3], cd);
        bs_sum<4>(ab, cd, U5);
        if constexpr (PU >= 5) bs_add(bigU, U5);
        else {
#pragma unroll
            for (int k = 0; k < PU; ++k) bigU[k] = U5[k];               // L = 4: one group only
        }
        // 8 spin words -> 4 planes
        const uint32_t x1 = xor3(sw[0], sw[1], sw[2]), y1 = maj3(sw[0], sw[1], sw[2]);
        const uint32_t x2 = xor3(sw[3], sw[4], sw[5]), y2 = maj3(sw[3], sw[4], sw[5]);
        const uint32_t x3 = xor3(x1, x2, sw[6]), y3 = maj3(x1, x2, sw[6]);
        const uint32_t ones = x3 ^ sw[7], y4 = x3 & sw[7];
        const uint32_t t1 = xor3(y1, y2, y3), f1 = maj3(y1, y2, y3);
        const uint32_t twos = t1 ^ y4, f2 = t1 & y4;
        const uint32_t M4[4] = {ones, twos, f1 ^ f2, f1 & f2};
        if constexpr (PM >= 4) bs_add(bigM, M4);
        else {
#pragma unroll
            for (int k = 0; k < PM; ++k) bigM[k] = M4[k];
        }
    }
    U = (int)bs_warp_total(bigU, PU, lane);
    M = 2 * (int)bs_warp_total(bigM, PM, lane) - N;
}

// ---- thread-block cluster helpers (split ladders): barrier over both CTAs, loads from the partner's shared memory
__device__ __forceinline__ void cluster_sync()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t dsmem_addr(const void *p, int rank)
{
    uint32_t a = (uint32_t)__cvta_generic_to_shared(p), r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(rank));
    return r;
}
__device__ __forceinline__ uint32_t ld_dsmem(const void *p, int rank)
{
    uint32_t v;
    asm volatile("ld.shared::cluster.u32 %0, [%1];" : "=r"(v) : "r"(dsmem_addr(p, rank)) : "memory");
    return v;
}
__device__ __forceinline__ uint4 ld_dsmem4(const void *p, int rank)
{
    uint4 v;
    asm volatile("ld.shared::cluster.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(dsmem_addr(p, rank)) : "memory");
    return v;
}

// ---- pieces of the exchange half sweep that one warp runs for its own pair of slots (pair and planar layouts)
// one word-site with the energy bookkeeping: new word and the three planes of its unsatisfied-bond count AFTER the update
template <bool BS>
__device__ __forceinline__ uint32_t update_word_energy(uint32_t sx, uint32_t amask, uint32_t u0, uint32_t u1, uint32_t u2, uint32_t u3,
                                                       uint32_t u4, uint32_t u5, uint32_t r, const SlotK &K, uint32_t one, uint32_t mone,
                                                       uint32_t (&wpl)[3])
{
    uint32_t n0, n1, n2;
    const uint32_t acc = accept_word<BS>(u0, u1, u2, u3, u4, u5, ~(sx ^ amask), r, K, one, mone, n0, n1, n2);
    // a flip turns n into 6 - n: bit 0 = n0; bit 1 set for n in {0, 3, 4}; bit 2 set for n in {0, 1, 2}
    const uint32_t f1 = (~n2 & ~(n1 ^ n0)) | (n2 & ~n1 & ~n0);
    const uint32_t f2 = ~n2 & ~(n1 & n0);
    wpl[0] = n0;
    wpl[1] = (acc & f1) | (~acc & n1);
    wpl[2] = (acc & f2) | (~acc & n2);
    return sx ^ acc;
}

// the four count planes of a quad and its eight spin words (four new, four of the other colour) -> the lane's running totals
template <int PU, int PM>
__device__ __forceinline__ void energy_accumulate(const uint32_t (&wpl)[4][3], const uint32_t (&outw)[4], const uint32_t (&othw)[4],
                                                  uint32_t (&aU)[PU], uint32_t (&aM)[PM])
{
    uint32_t ab[4], cd[4], U5[5];
    bs_sum<3>(wpl[0], wpl[1], ab);
    bs_sum<3>(wpl[2], wpl[3], cd);
    bs_sum<4>(ab, cd, U5);
    bs_add(aU, U5);
    const uint32_t x1 = xor3(outw[0], outw[1], outw[2]), y1 = maj3(outw[0], outw[1], outw[2]);
    const uint32_t x2 = xor3(outw[3], othw[0], othw[1]), y2 = maj3(outw[3], othw[0], othw[1]);
    const uint32_t x3 = xor3(x1, x2, othw[2]), y3 = maj3(x1, x2, othw[2]);
    const uint32_t ones = x3 ^ othw[3], y4 = x3 & othw[3];
    const uint32_t t1 = xor3(y1, y2, y3), g1 = maj3(y1, y2, y3);
    const uint32_t twos = t1 ^ y4, g2 = t1 & y4;
    const uint32_t M4[4] = {ones, twos, g1 ^ g2, g1 & g2};
    bs_add(aM, M4);
}

// which slots task `task` of exchange parity e1 covers: a pair (tA, tA + 1), or the slots without a partner this time
__device__ __forceinline__ void spw_task(int task, int e1, int NT, int &tA, int &tB, bool &paired)
{
    const int npairs = (NT - e1) / 2;
    const bool left_lo = e1 == 1, left_hi = ((NT - e1) & 1) != 0;
    paired = task < npairs;
    if (paired) { tA = e1 + 2 * task; tB = tA + 1; }
    else if (left_lo && left_hi) { tA = NT - 1; tB = 0; }
    else { tA = left_lo ? 0 : NT - 1; tB = tA; }
}
__device__ __forceinline__ int spw_ntask(int e1, int NT)
{
    return (NT - e1) / 2 + ((e1 == 1 || ((NT - e1) & 1) != 0) ? 1 : 0);
}

// after the warp's lanes walked both systems: per-lane totals, decision (R12), masked swap of the warp's own two systems,
// accepted-swap count, and (last sweep of the launch) the energies, permuted like the configurations
template <int L, int PU, int PM>
__device__ __forceinline__ void spw_finish(const LadderArgs &A, uint32_t *S, uint32_t *accs, const uint32_t (&aU0)[PU],
                                           const uint32_t (&aM0)[PM], const uint32_t (&aU1)[PU], const uint32_t (&aM1)[PM], int tA, int tB,
                                           bool paired, bool last, int lane, int w, int a, uint64_t exchange)
{
    constexpr int N = L * L * L;
    const Dims &d = A.d;
    __syncwarp();
    const int U0 = (int)bs_warp_total(aU0, PU, lane), M0 = 2 * (int)bs_warp_total(aM0, PM, lane) - N;
    const int U1 = (int)bs_warp_total(aU1, PU, lane), M1 = 2 * (int)bs_warp_total(aM1, PM, lane) - N;
    uint32_t mask = 0u;
    if (paired) {
        const int smp = w * 32 + lane;
        const double Et = __dsub_rn((double)(2 * U0 - 3 * N), __dmul_rn(A.h, (double)M0));
        const double Eu = __dsub_rn((double)(2 * U1 - 3 * N), __dmul_rn(A.h, (double)M1));
        const double x = __dmul_rn(__dsub_rn(A.tab[tA].beta, A.tab[tB].beta), __dsub_rn(Et, Eu));
        const uint4 r = philox_rk(0u, (uint32_t)exchange, (uint32_t)(smp + d.s_first), ctr3(4, a, tA), A.rk);
        const bool accept = (x >= 0.0) || ((uint64_t)r.x < dexp64(A.exp_tab, -x));
        mask = __ballot_sync(0xffffffffu, accept && smp < d.n_samples);
        if (lane == 0) accs[tA] += (uint32_t)__popc(mask);
        if (mask != 0u) {                             // masked swap (layout independent: the same position in both systems)
            for (int k = lane; k < N / 4; k += 32) {
                uint4 *X = reinterpret_cast<uint4 *>(S + tA * N) + k;
                uint4 *Y = reinterpret_cast<uint4 *>(S + tB * N) + k;
                uint4 xv = *X, yv = *Y;
                uint32_t dd;
                dd = (xv.x ^ yv.x) & mask; xv.x ^= dd; yv.x ^= dd;
                dd = (xv.y ^ yv.y) & mask; xv.y ^= dd; yv.y ^= dd;
                dd = (xv.z ^ yv.z) & mask; xv.z ^= dd; yv.z ^= dd;
                dd = (xv.w ^ yv.w) & mask; xv.w ^= dd; yv.w ^= dd;
                *X = xv;
                *Y = yv;
            }
        }
    }
    if (last) {
        const bool swp = (mask >> lane) & 1u;
        const size_t oA = ((size_t)(w * 32 + lane) * d.R + a) * d.NT + tA;
        A.U[oA] = (int64_t)(swp ? U1 : U0);
        A.M[oA] = swp ? M1 : M0;
        if (tB != tA) {
            const size_t oB = ((size_t)(w * 32 + lane) * d.R + a) * d.NT + tB;
            A.U[oB] = (int64_t)(swp ? U0 : U1);
            A.M[oB] = swp ? M0 : M1;
        }
    }
}

// PTM: 0 = the instantiation for launches without exchanges (all exchange code compiled out), 1 = exchanges by the recount
// path (any layout, split ladders), 2 = exchanges by the warp-per-pair half sweep (pair and planar layouts, A.use_spw)
template <int L, bool BS, int PTM>
__global__ void __launch_bounds__(Geo<L>::MAXT, Geo<L>::MINB) k_ladder_pmj(const __grid_constant__ LadderArgs A)
{
    constexpr bool PT = PTM != 0, SPW = PTM == 2;
    using G_ = Geo<L>;
    constexpr int Lh = G_::Lh, N = G_::N, H = G_::H, Q = G_::Q;
    extern __shared__ __align__(16) uint32_t smem[];
    const Dims &d = A.d;
    const int NT = d.NT;
    uint32_t *S = smem;                                   // [nt_res][2][H]: the slots this CTA owns
    uint32_t *Jsm = S + (size_t)A.nt_res * N;             // [2][3][H]
    uint2 *thr = reinterpret_cast<uint2 *>(Jsm + 3 * N);  // [NT][8]
    int *Uint = reinterpret_cast<int *>(thr + NT * 8);    // [NT][32]   exchange scratch (pt_every > 0 only)
    int *Mint = Uint + NT * 32;                           // [NT][32]
    uint32_t *masks = reinterpret_cast<uint32_t *>(Mint + NT * 32);   // [NT / 2 + 1]
    uint32_t *accs = masks + (NT / 2 + 1);                // [NT] accepted swaps of this CTA per lower slot
    // energy tables (use_tab): 16-byte aligned behind the scratch above
    uint4 *idxT = reinterpret_cast<uint4 *>((reinterpret_cast<uintptr_t>(accs + NT) + 15) & ~(uintptr_t)15);   // [H]
    uint32_t *JgT = reinterpret_cast<uint32_t *>(idxT + H);                                                     // [H][6]
    uint2 *spwT = reinterpret_cast<uint2 *>(idxT);        // [9][Q] byte offsets of the colour-1 quads (use_spw; instead of idxT / JgT)

    // this CTA: slots [tlo, tlo + ntl) of ladder `lad`.  CTAs [0, n_full) own whole ladders, the rest come in pairs that
    // share a ladder (first half of the slots rounded up, second half)
    int lad = blockIdx.x, tlo = 0, ntl = NT, half = 0;
    if ((int)blockIdx.x >= A.n_full) {
        const int idx = (int)blockIdx.x - A.n_full;
        lad = A.n_full + (idx >> 1);
        half = idx & 1;
        const int nt0 = (NT + 1) / 2;
        tlo = half ? nt0 : 0;
        ntl = half ? NT - nt0 : nt0;
    }
    const bool split_pt = PT && A.split != 0;              // the partner CTA (cluster rank 1 - half) holds the other slots
    const int w = lad / d.R, a = lad % d.R;
    const int tid = threadIdx.x, nthr = blockDim.x;
    uint32_t *gS = A.spins + ((size_t)(w * d.R + a) * NT + tlo) * N;
    uint32_t *gOut = A.spins_out + ((size_t)(w * d.R + a) * NT + tlo) * N;
    const uint32_t *gJ = A.J + (size_t)w * 3 * N;

    // ---- load the ladder, the couplings and the threshold constants
    {
        const uint4 *src = reinterpret_cast<const uint4 *>(gS);
        const uint4 *js = reinterpret_cast<const uint4 *>(gJ);
        if constexpr (G_::PAIR) {                              // quad i of a colour block -> its low and high pair
            uint2 *dst = reinterpret_cast<uint2 *>(S), *jd = reinterpret_cast<uint2 *>(Jsm);
            for (int i = tid; i < ntl * N / 4; i += nthr) {
                const int blk = i / Q, qd = i - blk * Q;
                const uint4 v = src[i];
                dst[blk * (2 * Q) + qd] = make_uint2(v.x, v.y);
                dst[blk * (2 * Q) + Q + qd] = make_uint2(v.z, v.w);
            }
            for (int i = tid; i < 3 * N / 4; i += nthr) {
                const int blk = i / Q, qd = i - blk * Q;
                const uint4 v = js[i];
                jd[blk * (2 * Q) + qd] = make_uint2(v.x, v.y);
                jd[blk * (2 * Q) + Q + qd] = make_uint2(v.z, v.w);
            }
        } else if constexpr (G_::PLANAR) {                      // quad i of a colour block -> word e to array e
            for (int i = tid; i < ntl * N / 4; i += nthr) {
                const int blk = i / Q, qd = i - blk * Q;
                const uint4 v = src[i];
                uint32_t *dst = S + blk * H + qd;
                dst[0] = v.x; dst[Q] = v.y; dst[2 * Q] = v.z; dst[3 * Q] = v.w;
            }
            for (int i = tid; i < 3 * N / 4; i += nthr) {
                const int blk = i / Q, qd = i - blk * Q;
                const uint4 v = js[i];
                uint32_t *dst = Jsm + blk * H + qd;
                dst[0] = v.x; dst[Q] = v.y; dst[2 * Q] = v.z; dst[3 * Q] = v.w;
            }
        } else {
            uint4 *dst = reinterpret_cast<uint4 *>(S);
            for (int i = tid; i < ntl * N / 4; i += nthr) dst[i] = src[i];
            uint4 *jd = reinterpret_cast<uint4 *>(Jsm);
            for (int i = tid; i < 3 * N / 4; i += nthr) jd[i] = js[i];
        }
        for (int t = tid; t < NT; t += nthr) {                 // acceptance constants (SlotK of sg_accept.cuh)
            uint32_t lo[7], hi[7], kw[10];
            for (int c = 0; c < 7; ++c) {
                const uint2 v = A.tab[t].c64[c];               // (0 - thr) as 64 bits
                lo[c] = v.x;
                hi[c] = v.y;
            }
            slotk_words<BS>(lo, hi, kw);
            uint4 *k4 = reinterpret_cast<uint4 *>(thr + t * 8);
            k4[0] = make_uint4(kw[0], kw[1], kw[2], kw[3]);
            k4[1] = make_uint4(kw[4], kw[5], kw[6], kw[7]);
            k4[2] = make_uint4(kw[8], kw[9], 0u, 0u);
        }
        for (int t = tid; t < NT; t += nthr) accs[t] = 0u;
    }
    __syncthreads();
    if (PT && !SPW && A.use_tab && A.pt_every > 0) {      // neighbour indices and couplings of the colour-0 sites, once per launch
        const uint32_t *J0 = Jsm, *J1 = Jsm + 3 * H;
        for (int n = tid; n < H; n += nthr) {
            const int row = n / Lh, m = n - row * Lh;
            const int z = row / L, y = row - z * L;
            const int p = (y + z) & 1;
            const int sd = row * Lh + (p ? (m + 1 == Lh ? 0 : m + 1) : (m == 0 ? Lh - 1 : m - 1));
            const int xp = p ? sd : n, xm = p ? n : sd;
            const int yp = (z * L + (y + 1 == L ? 0 : y + 1)) * Lh + m, ym = (z * L + (y == 0 ? L - 1 : y - 1)) * Lh + m;
            const int zp = ((z + 1 == L ? 0 : z + 1) * L + y) * Lh + m, zm = ((z == 0 ? L - 1 : z - 1) * L + y) * Lh + m;
            constexpr auto P = G_::pos;
            idxT[n] = make_uint4((uint32_t)P(xp) | ((uint32_t)P(xm) << 16), (uint32_t)P(yp) | ((uint32_t)P(ym) << 16),
                                 (uint32_t)P(zp) | ((uint32_t)P(zm) << 16), (uint32_t)P(n));
            uint32_t *g = JgT + 6 * n;
            g[0] = J0[P(n)];          g[1] = J1[P(xm)];
            g[2] = J0[H + P(n)];      g[3] = J1[H + P(ym)];
            g[4] = J0[2 * H + P(n)];  g[5] = J1[2 * H + P(zm)];
        }
        __syncthreads();
    }

    if constexpr (G_::PAIR) {
        if (SPW && A.pt_every > 0) {
            // Offsets (bytes) for the colour-1 half sweep that precedes an exchange, where a WARP owns two systems and its
            // lanes walk the quads, so nothing can be hoisted into registers.  Per pair hh of quad qd, relative to the
            // other-colour block of the system: +y, -y, +z, -z neighbour pairs and the two side words; relative to the
            // couplings: the pair of slot 0 and the two words of slot 1 (see the block-item path below for the selection).
            constexpr int Q2 = 2 * Q;
            for (int qd = tid; qd < Q; qd += nthr) {
#pragma unroll
                for (int hh = 0; hh < 2; ++hh) {
                    const int n = 4 * qd + 2 * hh, o = hh * Q2 + 2 * qd;
                    const int row = n / Lh, m = n - row * Lh;
                    const int z = row / L, y = row - z * L;
                    const int p = (1 + y + z) & 1;
                    const int yp = (z * L + (y + 1 == L ? 0 : y + 1)) * Lh + m;
                    const int ym = (z * L + (y == 0 ? L - 1 : y - 1)) * Lh + m;
                    const int zp = ((z + 1 == L ? 0 : z + 1) * L + y) * Lh + m;
                    const int zm = ((z == 0 ? L - 1 : z - 1) * L + y) * Lh + m;
                    const int sdn = G_::pos(p ? (m + 2 == Lh ? row * Lh : n + 2) : (m == 0 ? row * Lh + Lh - 1 : n - 1));
                    constexpr int JOWN = 3 * H, JOTH = 0;               // colour 1 owns the second coupling block
                    uint32_t e[9];
                    e[0] = 4u * G_::pos(yp); e[1] = 4u * G_::pos(ym); e[2] = 4u * G_::pos(zp); e[3] = 4u * G_::pos(zm);
                    e[4] = 4u * (p ? o + 1 : sdn);
                    e[5] = 4u * (p ? sdn : o);
                    e[6] = 4u * (p ? JOTH + o : JOWN + o);
                    e[7] = 4u * (p ? JOWN + o : JOTH + sdn);
                    e[8] = 4u * (p ? JOWN + o + 1 : JOTH + o);
                    uint32_t *T = reinterpret_cast<uint32_t *>(spwT);   // word k of pair hh of quad qd: T[((k * Q) + qd) * 2 + hh]
#pragma unroll
                    for (int k = 0; k < 9; ++k) T[(k * Q + qd) * 2 + hh] = e[k];
                }
            }
            __syncthreads();
        }
    }

    if constexpr (G_::PLANAR) {
        if (SPW && A.pt_every > 0) {
            // planar layout, exchange half sweep by one warp per pair of slots: positions of the six neighbours and the six
            // coupling words of every colour-1 site, [element e][neighbour k][quad] (unit-stride over the lanes)
            uint32_t *ixT = reinterpret_cast<uint32_t *>(spwT), *JgS = ixT + 24 * Q;
            const uint32_t *Jown = Jsm + 3 * H, *Joth = Jsm;          // colour 1 owns the second coupling block
            for (int i = tid; i < 4 * Q; i += nthr) {
                const int e = i / Q, qd = i - e * Q;
                const int n = 4 * qd + e;
                const int row = n / Lh, m = n - row * Lh;
                const int z = row / L, y = row - z * L;
                const int p = (1 + y + z) & 1;
                const int sd = row * Lh + (p ? (m + 1 == Lh ? 0 : m + 1) : (m == 0 ? Lh - 1 : m - 1));
                const int yp = (z * L + (y + 1 == L ? 0 : y + 1)) * Lh + m;
                const int ym = (z * L + (y == 0 ? L - 1 : y - 1)) * Lh + m;
                const int zp = ((z + 1 == L ? 0 : z + 1) * L + y) * Lh + m;
                const int zm = ((z == 0 ? L - 1 : z - 1) * L + y) * Lh + m;
                constexpr auto P = G_::pos;
                const int ixv[6] = {P(n), P(sd), P(yp), P(ym), P(zp), P(zm)};
                const uint32_t jv[6] = {p ? Joth[P(n)] : Jown[P(n)], p ? Jown[P(n)] : Joth[P(sd)], Jown[H + P(n)], Joth[H + P(ym)],
                                        Jown[2 * H + P(n)], Joth[2 * H + P(zm)]};
#pragma unroll
                for (int k = 0; k < 6; ++k) {
                    ixT[(e * 6 + k) * Q + qd] = (uint32_t)ixv[k];
                    JgS[(e * 6 + k) * Q + qd] = jv[k];
                }
            }
            __syncthreads();
        }
    }

    const int q = tid % Q, g = tid / Q;
    const bool active = g < A.G;
    const uint32_t amask = d.neg_h ? 0xffffffffu : 0u;     // a = s ^ amask ; na = ~a
    const uint32_t wglob = (uint32_t)(w + (d.s_first >> 5));
    uint64_t exchange = A.exchange0;

    for (int sw = 0; sw < A.n_sweeps; ++sw) {
#pragma unroll 1
        for (int colour = 0; colour < 2; ++colour) {
            if constexpr (G_::VEC) {
                // rows are whole quads: every neighbour of a quad is an aligned 128-bit access, except the one word beyond
                // each end of the quad (side)
                constexpr int QR = G_::QR, NBV = Q / 32;
                constexpr int PU = NBV * 24 < 32 ? 5 : NBV * 24 < 64 ? 6 : NBV * 24 < 128 ? 7 : NBV * 24 < 256 ? 8 : 9;
                constexpr int PM = NBV * 8 < 16 ? 4 : NBV * 8 < 32 ? 5 : NBV * 8 < 64 ? 6 : NBV * 8 < 128 ? 7 : 8;
                static_assert(Q % 32 == 0 && NBV * 24 < 512 && NBV * 8 < 256, "plane counts");
                const uint32_t time = 2u * (A.sweep0 + (uint32_t)sw) + (uint32_t)colour;
                const uint32_t *Jown = Jsm + (colour * 3) * H;
                const uint32_t *Joth = Jsm + ((1 - colour) * 3) * H;
                int q_yp = 0, q_ym = 0, q_zp = 0, q_zm = 0, side[4] = {0, 0, 0, 0};
                uint32_t JA[4], JB[4], Jyp[4], Jym[4], Jzp[4], Jzm[4];
                // neighbour quads and the 24 coupling words of quad qx (shared by all systems handled with it)
                auto setup = [&](const int qx) {
                    const int r = qx / QR, kq = qx % QR;
                    const int y = r % L, z = r / L;
                    const int p = (colour + y + z) & 1;
                    q_yp = (y + 1 == L) ? qx - (L - 1) * QR : qx + QR;
                    q_ym = (y == 0) ? qx + (L - 1) * QR : qx - QR;
                    q_zp = (z + 1 == L) ? qx - (L - 1) * L * QR : qx + L * QR;
                    q_zm = (z == 0) ? qx + (L - 1) * L * QR : qx - L * QR;
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        const int m = 4 * kq + e;
                        const int ms = p ? (m + 1 == Lh ? 0 : m + 1) : (m == 0 ? Lh - 1 : m - 1);
                        side[e] = r * Lh + ms;
                    }
                    const uint4 jx = reinterpret_cast<const uint4 *>(Jown)[qx];
                    const uint4 jox = reinterpret_cast<const uint4 *>(Joth)[qx];
                    const uint4 jy = reinterpret_cast<const uint4 *>(Jown + H)[qx];
                    const uint4 joy = reinterpret_cast<const uint4 *>(Joth + H)[q_ym];
                    const uint4 jz = reinterpret_cast<const uint4 *>(Jown + 2 * H)[qx];
                    const uint4 joz = reinterpret_cast<const uint4 *>(Joth + 2 * H)[q_zm];
                    const uint32_t jxv[4] = {jx.x, jx.y, jx.z, jx.w}, joxv[4] = {jox.x, jox.y, jox.z, jox.w};
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        // bond to the neighbour at the same compact index / at the side index
                        JA[e] = p ? joxv[e] : jxv[e];
                        JB[e] = p ? jxv[e] : Joth[side[e]];
                    }
                    Jyp[0] = jy.x; Jyp[1] = jy.y; Jyp[2] = jy.z; Jyp[3] = jy.w;
                    Jym[0] = joy.x; Jym[1] = joy.y; Jym[2] = joy.z; Jym[3] = joy.w;
                    Jzp[0] = jz.x; Jzp[1] = jz.y; Jzp[2] = jz.z; Jzp[3] = jz.w;
                    Jzm[0] = joz.x; Jzm[1] = joz.y; Jzm[2] = joz.z; Jzm[3] = joz.w;
                };
                // quad qx of slot t (Sa / So = its own / the other colour block); en: with the energy bookkeeping
                auto vitem = [&](const bool en, const int qx, const int t, uint32_t *__restrict__ Sa, const uint32_t *__restrict__ So,
                                 uint32_t (&aU)[PU], uint32_t (&aM)[PM]) {
                    const uint4 sv = reinterpret_cast<const uint4 *>(Sa)[qx];
                    const uint4 o0 = reinterpret_cast<const uint4 *>(So)[qx];
                    const uint4 oyp = reinterpret_cast<const uint4 *>(So)[q_yp];
                    const uint4 oym = reinterpret_cast<const uint4 *>(So)[q_ym];
                    const uint4 ozp = reinterpret_cast<const uint4 *>(So)[q_zp];
                    const uint4 ozm = reinterpret_cast<const uint4 *>(So)[q_zm];
                    const uint32_t os[4] = {So[side[0]], So[side[1]], So[side[2]], So[side[3]]};
                    const uint4 r4 = philox_rk((uint32_t)qx, time, wglob, ctr3(3, a, t), A.rk);
                    SlotK K;
                    {
                        const uint4 *k4 = reinterpret_cast<const uint4 *>(thr + t * 8);
                        const uint4 k0 = k4[0], k1 = k4[1], k2 = k4[2];
                        K.lo[0] = k0.x; K.lo[1] = k0.y; K.lo[2] = k0.z; K.lo[3] = k0.w;
                        K.lo[4] = k1.x; K.lo[5] = k1.y; K.lo[6] = k1.z; K.b3c = k1.w;
                        K.nc = k2.x; K.ec = k2.y;
                    }
                    const uint32_t s[4] = {sv.x, sv.y, sv.z, sv.w};
                    const uint32_t rr[4] = {r4.x, r4.y, r4.z, r4.w};
                    const uint32_t v0[4] = {o0.x, o0.y, o0.z, o0.w}, vyp[4] = {oyp.x, oyp.y, oyp.z, oyp.w};
                    const uint32_t vym[4] = {oym.x, oym.y, oym.z, oym.w}, vzp[4] = {ozp.x, ozp.y, ozp.z, ozp.w};
                    const uint32_t vzm[4] = {ozm.x, ozm.y, ozm.z, ozm.w};
                    uint32_t out[4];
                    if (en) {                                      // (a literal at both call sites)
                        uint32_t wpl[4][3];
#pragma unroll
                        for (int e = 0; e < 4; ++e)
                            out[e] = update_word_energy<BS>(s[e], amask, xor3(s[e], v0[e], JA[e]), xor3(s[e], os[e], JB[e]),
                                                            xor3(s[e], vyp[e], Jyp[e]), xor3(s[e], vym[e], Jym[e]),
                                                            xor3(s[e], vzp[e], Jzp[e]), xor3(s[e], vzm[e], Jzm[e]), rr[e], K, A.one,
                                                            A.mone, wpl[e]);
                        energy_accumulate(wpl, out, v0, aU, aM);
                    } else {
#pragma unroll
                        for (int e = 0; e < 4; ++e)
                            out[e] = flip_word_k<BS>(s[e], amask, xor3(s[e], v0[e], JA[e]), xor3(s[e], os[e], JB[e]),
                                                     xor3(s[e], vyp[e], Jyp[e]), xor3(s[e], vym[e], Jym[e]),
                                                     xor3(s[e], vzp[e], Jzp[e]), xor3(s[e], vzm[e], Jzm[e]), rr[e], K, A.one,
                                                     A.mone);
                    }
                    reinterpret_cast<uint4 *>(Sa)[qx] = make_uint4(out[0], out[1], out[2], out[3]);
                };
                const bool spw_now = SPW && colour == 1 && A.pt_every > 0 &&
                                     ((uint64_t)A.sweep0 + (uint64_t)sw + 1) % (uint64_t)A.pt_every == 0;
                if (spw_now) {
                    // ---- colour-1 half sweep + exchange, one WARP per pair of neighbouring slots (see the pair layout below)
                    const int lane_ = tid & 31, warp_ = tid >> 5, NW = nthr >> 5;
                    const int e1 = (int)(exchange & 1u);
                    const int ntask = spw_ntask(e1, NT);
                    const bool last = sw == A.n_sweeps - 1;
                    for (int task = warp_; task < ntask; task += NW) {
                        int tA, tB;
                        bool paired;
                        spw_task(task, e1, NT, tA, tB, paired);
                        const bool two = tB != tA;
                        const int offB = (tB - tA) * N;
                        uint32_t *SaA = S + tA * N + H;
                        const uint32_t *SoA = S + tA * N;
                        uint32_t aU0[PU], aM0[PM], aU1[PU], aM1[PM];
#pragma unroll
                        for (int k = 0; k < PU; ++k) aU0[k] = aU1[k] = 0u;
#pragma unroll
                        for (int k = 0; k < PM; ++k) aM0[k] = aM1[k] = 0u;
#pragma unroll 1
                        for (int kb = 0; kb < NBV; ++kb) {
                            const int qx = 32 * kb + lane_;
                            setup(qx);
                            vitem(true, qx, tA, SaA, SoA, aU0, aM0);
                            if (two) vitem(true, qx, tB, SaA + offB, SoA + offB, aU1, aM1);
                        }
                        spw_finish<L>(A, S, accs, aU0, aM0, aU1, aM1, tA, tB, paired, last, lane_, w, a, exchange);
                    }
                } else if (active) {
                    uint32_t dU[PU], dM[PM];                       // (unused by the instantiation without bookkeeping)
                    setup(q);
#pragma unroll 1
                    for (int tl = g; tl < ntl; tl += A.G)
                        vitem(false, q, tlo + tl, S + tl * N + colour * H, S + tl * N + (1 - colour) * H, dU, dM);
                }
            }
            if constexpr (!G_::VEC) {
                // generic lattice (rows of L/2 words are not whole quads).  Work item = (block of 32 quads, system); the
                // NB * NT items of a half sweep are dealt out in contiguous ranges so that the four warp schedulers get the
                // same number of items (warp w runs on scheduler w % 4).  Per-element neighbour indices and the 24 coupling
                // words of the quad are computed / loaded when the block of a warp changes (at most twice per half sweep).
                constexpr int NB = (Q + 31) / 32;
                const uint32_t time = 2u * (A.sweep0 + (uint32_t)sw) + (uint32_t)colour;
                const uint32_t *Jown = Jsm + (colour * 3) * H;
                const uint32_t *Joth = Jsm + ((1 - colour) * 3) * H;
                const int lane_ = tid & 31, warp_ = tid >> 5, NW = nthr >> 5;
                const int rank = (warp_ & 3) * (NW >> 2) + (warp_ >> 2);
                const int I = NB * ntl;                  // (ntl = NT unless this CTA owns half a ladder)
                const int i1 = (rank + 1) * I / NW;
                int qq = 0;
                bool qa = false;
                if constexpr (G_::PAIR) {
                    // pair layout (Geo::PAIR): per 64-bit pair h of the quad, the positions of its +-y / +-z neighbour
                    // pairs and of the ONE word beyond the pair that its side (x) neighbours need, the row parity as a
                    // mask, and the 24 coupling words of the quad
                    constexpr int Q2 = 2 * Q;
                    int ip[2][6];
                    uint32_t Jq[4][6];
                    // one work item: system t of the current block (Sa / So = its own / the other colour block)
                    auto item = [&](const int t, uint32_t *__restrict__ Sa, const uint32_t *__restrict__ So) {
                        const uint4 r4 = philox_rk((uint32_t)qq, time, wglob, ctr3(3, a, t), A.rk);
                        SlotK K;
                        {
                            const uint4 *k4 = reinterpret_cast<const uint4 *>(thr + t * 8);
                            const uint4 k0 = k4[0], k1 = k4[1], k2 = k4[2];
                            K.lo[0] = k0.x; K.lo[1] = k0.y; K.lo[2] = k0.z; K.lo[3] = k0.w;
                            K.lo[4] = k1.x; K.lo[5] = k1.y; K.lo[6] = k1.z; K.b3c = k1.w;
                            K.nc = k2.x; K.ec = k2.y;
                        }
                        const uint32_t rr[4] = {r4.x, r4.y, r4.z, r4.w};
#pragma unroll
                        for (int hh = 0; hh < 2; ++hh) {
                            const int o = hh * Q2 + 2 * qq;
                            const uint2 sv = *reinterpret_cast<const uint2 *>(Sa + o);
                            const uint2 a0 = *reinterpret_cast<const uint2 *>(So + o);
                            const uint2 vyp = *reinterpret_cast<const uint2 *>(So + ip[hh][0]);
                            const uint2 vym = *reinterpret_cast<const uint2 *>(So + ip[hh][1]);
                            const uint2 vzp = *reinterpret_cast<const uint2 *>(So + ip[hh][2]);
                            const uint2 vzm = *reinterpret_cast<const uint2 *>(So + ip[hh][3]);
                            const uint32_t sd0 = So[ip[hh][4]], sd1 = So[ip[hh][5]];
                            const int e0 = 2 * hh, e1 = 2 * hh + 1;
                            const uint32_t o0 = flip_word_k<BS>(sv.x, amask, xor3(sv.x, a0.x, Jq[e0][0]), xor3(sv.x, sd0, Jq[e0][1]),
                                                                xor3(sv.x, vyp.x, Jq[e0][2]), xor3(sv.x, vym.x, Jq[e0][3]),
                                                                xor3(sv.x, vzp.x, Jq[e0][4]), xor3(sv.x, vzm.x, Jq[e0][5]), rr[e0], K,
                                                                A.one, A.mone);
                            const uint32_t o1 = flip_word_k<BS>(sv.y, amask, xor3(sv.y, a0.y, Jq[e1][0]), xor3(sv.y, sd1, Jq[e1][1]),
                                                                xor3(sv.y, vyp.y, Jq[e1][2]), xor3(sv.y, vym.y, Jq[e1][3]),
                                                                xor3(sv.y, vzp.y, Jq[e1][4]), xor3(sv.y, vzm.y, Jq[e1][5]), rr[e1], K,
                                                                A.one, A.mone);
                            if (qa) *reinterpret_cast<uint2 *>(Sa + o) = make_uint2(o0, o1);
                        }
                    };
                    // The same work item with the energy bookkeeping of the exchange step (colour 1 only): U = sum over the
                    // colour-1 sites of their unsatisfied-bond counts AFTER the update (every bond has one colour-1 end; a flip
                    // turns n into 6 - n), spin count = the four new words + the four other-colour words at the same compact
                    // index; both added to the lane's running bit-sliced totals.
                    constexpr int PU = NB * 24 < 32 ? 5 : NB * 24 < 64 ? 6 : NB * 24 < 128 ? 7 : NB * 24 < 256 ? 8 : 9;
                    constexpr int PM = NB * 8 < 16 ? 4 : NB * 8 < 32 ? 5 : NB * 8 < 64 ? 6 : 7;
                    static_assert(NB * 24 < 512 && NB * 8 < 128, "plane counts");
                    auto itemE = [&](const int t, uint32_t *__restrict__ Sa, const uint32_t *__restrict__ So, uint32_t (&aU)[PU],
                                     uint32_t (&aM)[PM]) {
                        const uint4 r4 = philox_rk((uint32_t)qq, time, wglob, ctr3(3, a, t), A.rk);
                        SlotK K;
                        {
                            const uint4 *k4 = reinterpret_cast<const uint4 *>(thr + t * 8);
                            const uint4 k0 = k4[0], k1 = k4[1], k2 = k4[2];
                            K.lo[0] = k0.x; K.lo[1] = k0.y; K.lo[2] = k0.z; K.lo[3] = k0.w;
                            K.lo[4] = k1.x; K.lo[5] = k1.y; K.lo[6] = k1.z; K.b3c = k1.w;
                            K.nc = k2.x; K.ec = k2.y;
                        }
                        const uint32_t rr[4] = {r4.x, r4.y, r4.z, r4.w};
                        uint32_t wpl[4][3], outw[4], othw[4];
#pragma unroll
                        for (int hh = 0; hh < 2; ++hh) {
                            const int o = hh * Q2 + 2 * qq;
                            const uint2 sv = *reinterpret_cast<const uint2 *>(Sa + o);
                            const uint2 a0 = *reinterpret_cast<const uint2 *>(So + o);
                            const uint2 vyp = *reinterpret_cast<const uint2 *>(So + ip[hh][0]);
                            const uint2 vym = *reinterpret_cast<const uint2 *>(So + ip[hh][1]);
                            const uint2 vzp = *reinterpret_cast<const uint2 *>(So + ip[hh][2]);
                            const uint2 vzm = *reinterpret_cast<const uint2 *>(So + ip[hh][3]);
                            const uint32_t sdw[2] = {So[ip[hh][4]], So[ip[hh][5]]};
                            const uint32_t sw2[2] = {sv.x, sv.y}, a02[2] = {a0.x, a0.y}, yp2[2] = {vyp.x, vyp.y}, ym2[2] = {vym.x, vym.y};
                            const uint32_t zp2[2] = {vzp.x, vzp.y}, zm2[2] = {vzm.x, vzm.y};
#pragma unroll
                            for (int j = 0; j < 2; ++j) {
                                const int e = 2 * hh + j;
                                const uint32_t sx = sw2[j];
                                outw[e] = update_word_energy<BS>(sx, amask, xor3(sx, a02[j], Jq[e][0]), xor3(sx, sdw[j], Jq[e][1]),
                                                                 xor3(sx, yp2[j], Jq[e][2]), xor3(sx, ym2[j], Jq[e][3]),
                                                                 xor3(sx, zp2[j], Jq[e][4]), xor3(sx, zm2[j], Jq[e][5]), rr[e], K,
                                                                 A.one, A.mone, wpl[e]);
                                othw[e] = a02[j];
                            }
                            *reinterpret_cast<uint2 *>(Sa + o) = make_uint2(outw[2 * hh], outw[2 * hh + 1]);
                        }
                        energy_accumulate(wpl, outw, othw, aU, aM);
                    };
                    const bool pt_due_now = SPW && colour == 1 && A.pt_every > 0 &&
                                            ((uint64_t)A.sweep0 + (uint64_t)sw + 1) % (uint64_t)A.pt_every == 0;
                    if (pt_due_now) {
                        // ---- colour-1 half sweep + exchange, one WARP per pair of neighbouring slots: the lanes walk the quads
                        // of both systems (offsets and couplings from the table / shared memory), keep the energy counts in
                        // registers, and the warp then decides and swaps its own two systems: no pass over the ladder and no
                        // CTA barrier between the half sweep, the decisions and the swaps.
                        const int e1 = (int)(exchange & 1u);
                        const int ntask = spw_ntask(e1, NT);
                        const bool last = sw == A.n_sweeps - 1;
                        for (int task = warp_; task < ntask; task += NW) {
                            int tA, tB;
                            bool paired;
                            spw_task(task, e1, NT, tA, tB, paired);
                            const bool two = tB != tA;
                            const int offB = (tB - tA) * N;
                            uint32_t *SaA = S + tA * N + H;
                            const uint32_t *SoA = S + tA * N;
                            uint32_t aU0[PU], aM0[PM], aU1[PU], aM1[PM];
#pragma unroll
                            for (int k = 0; k < PU; ++k) aU0[k] = aU1[k] = 0u;
#pragma unroll
                            for (int k = 0; k < PM; ++k) aM0[k] = aM1[k] = 0u;
#pragma unroll 1
                            for (int kb = 0; kb < NB; ++kb) {
                                qq = 32 * kb + lane_;
                                qa = true;
                                if (qq < Q) {
                                    uint2 tk[9];                              // entry k of both pairs of the quad: one 64-bit load
#pragma unroll
                                    for (int k = 0; k < 9; ++k) tk[k] = spwT[k * Q + qq];
#pragma unroll
                                    for (int hh = 0; hh < 2; ++hh) {
                                        const int o = hh * Q2 + 2 * qq;
                                        uint32_t ee[9];
#pragma unroll
                                        for (int k = 0; k < 9; ++k) ee[k] = hh ? tk[k].y : tk[k].x;
#pragma unroll
                                        for (int k = 0; k < 6; ++k) ip[hh][k] = (int)(ee[k] >> 2);
                                        const char *Jb = reinterpret_cast<const char *>(Jsm);
                                        const uint2 j0 = *reinterpret_cast<const uint2 *>(Jb + ee[6]);
                                        const uint32_t j1a = *reinterpret_cast<const uint32_t *>(Jb + ee[7]);
                                        const uint32_t j1b = *reinterpret_cast<const uint32_t *>(Jb + ee[8]);
                                        const uint2 jy = *reinterpret_cast<const uint2 *>(Jsm + 3 * H + H + o);
                                        const uint2 joy = *reinterpret_cast<const uint2 *>(Jb + 4 * H + ee[1]);
                                        const uint2 jz = *reinterpret_cast<const uint2 *>(Jsm + 3 * H + 2 * H + o);
                                        const uint2 joz = *reinterpret_cast<const uint2 *>(Jb + 8 * H + ee[3]);
                                        Jq[2 * hh][0] = j0.x;   Jq[2 * hh + 1][0] = j0.y;
                                        Jq[2 * hh][1] = j1a;    Jq[2 * hh + 1][1] = j1b;
                                        Jq[2 * hh][2] = jy.x;   Jq[2 * hh + 1][2] = jy.y;
                                        Jq[2 * hh][3] = joy.x;  Jq[2 * hh + 1][3] = joy.y;
                                        Jq[2 * hh][4] = jz.x;   Jq[2 * hh + 1][4] = jz.y;
                                        Jq[2 * hh][5] = joz.x;  Jq[2 * hh + 1][5] = joz.y;
                                    }
                                    itemE(tA, SaA, SoA, aU0, aM0);
                                    if (two) itemE(tB, SaA + offB, SoA + offB, aU1, aM1);
                                }
                            }
                            spw_finish<L>(A, S, accs, aU0, aM0, aU1, aM1, tA, tB, paired, last, lane_, w, a, exchange);
                        }
                    } else {
                    const int i0 = rank * I / NW;
                    int b = i0 / ntl, t = i0 - b * ntl;         // t: index among this CTA's slots
#pragma unroll 1
                    for (int i = i0; i < i1;) {
                        if (t == ntl) { t = 0; ++b; }
                        {
                            qq = 32 * b + lane_;
                            qa = qq < Q;
                            if (!qa) qq = Q - 1;
#pragma unroll
                            for (int hh = 0; hh < 2; ++hh) {
                                const int n = 4 * qq + 2 * hh, o = hh * Q2 + 2 * qq;
                                const int row = n / Lh, m = n - row * Lh;
                                const int z = row / L, y = row - z * L;
                                const int p = (colour + y + z) & 1;
                                const int yp = (z * L + (y + 1 == L ? 0 : y + 1)) * Lh + m;
                                const int ym = (z * L + (y == 0 ? L - 1 : y - 1)) * Lh + m;
                                const int zp = ((z + 1 == L ? 0 : z + 1) * L + y) * Lh + m;
                                const int zm = ((z == 0 ? L - 1 : z - 1) * L + y) * Lh + m;
                                // p: the side neighbours are m + 1 (the pair's own second word, and the word after the pair);
                                // else m - 1 (the word before the pair, and the pair's own first word); periodic in the row
                                const int sdn = G_::pos(p ? (m + 2 == Lh ? row * Lh : n + 2) : (m == 0 ? row * Lh + Lh - 1 : n - 1));
                                ip[hh][0] = G_::pos(yp); ip[hh][1] = G_::pos(ym); ip[hh][2] = G_::pos(zp); ip[hh][3] = G_::pos(zm);
                                ip[hh][4] = p ? o + 1 : sdn;
                                ip[hh][5] = p ? sdn : o;
                                const uint2 jx = *reinterpret_cast<const uint2 *>(Jown + o);
                                const uint2 jox = *reinterpret_cast<const uint2 *>(Joth + o);
                                const uint2 jy = *reinterpret_cast<const uint2 *>(Jown + H + o);
                                const uint2 joy = *reinterpret_cast<const uint2 *>(Joth + H + ip[hh][1]);
                                const uint2 jz = *reinterpret_cast<const uint2 *>(Jown + 2 * H + o);
                                const uint2 joz = *reinterpret_cast<const uint2 *>(Joth + 2 * H + ip[hh][3]);
                                const uint32_t jsd = Joth[sdn];
                                // slot 0: the x-neighbour at the same compact index (its bond if p, own bond else); slot 1: the side one
                                Jq[2 * hh][0] = p ? jox.x : jx.x;      Jq[2 * hh + 1][0] = p ? jox.y : jx.y;
                                Jq[2 * hh][1] = p ? jx.x : jsd;        Jq[2 * hh + 1][1] = p ? jx.y : jox.x;
                                Jq[2 * hh][2] = jy.x;   Jq[2 * hh + 1][2] = jy.y;
                                Jq[2 * hh][3] = joy.x;  Jq[2 * hh + 1][3] = joy.y;
                                Jq[2 * hh][4] = jz.x;   Jq[2 * hh + 1][4] = jz.y;
                                Jq[2 * hh][5] = joz.x;  Jq[2 * hh + 1][5] = joz.y;
                            }
                        }
                        // the systems t .. tend - 1 of this block, two per trip (the second one at a compile-time offset)
                        const int tend = min(ntl, t + (i1 - i));
                        i += tend - t;
                        uint32_t *Sa = S + t * N + colour * H;
                        const uint32_t *So = S + t * N + (1 - colour) * H;
#pragma unroll 1
                        for (; t + 1 < tend; t += 2, Sa += 2 * N, So += 2 * N) {
                            item(tlo + t, Sa, So);
                            item(tlo + t + 1, Sa + N, So + N);
                        }
                        if (t < tend) {
                            item(tlo + t, Sa, So);
                            ++t;
                        }
                    }
                    }
                } else if (SPW && colour == 1 && A.pt_every > 0 &&
                           ((uint64_t)A.sweep0 + (uint64_t)sw + 1) % (uint64_t)A.pt_every == 0) {
                    // ---- planar layout: colour-1 half sweep + exchange, one WARP per pair of neighbouring slots (as in the
                    // pair layout above; neighbour positions and couplings from the tables built at the start of the launch)
                    constexpr int PU = NB * 24 < 32 ? 5 : NB * 24 < 64 ? 6 : NB * 24 < 128 ? 7 : NB * 24 < 256 ? 8 : 9;
                    constexpr int PM = NB * 8 < 16 ? 4 : NB * 8 < 32 ? 5 : NB * 8 < 64 ? 6 : 7;
                    static_assert(NB * 24 < 512 && NB * 8 < 128, "plane counts");
                    const uint32_t *ixT = reinterpret_cast<const uint32_t *>(spwT), *JgS = ixT + 24 * Q;
                    const int e1 = (int)(exchange & 1u);
                    const int ntask = spw_ntask(e1, NT);
                    const bool last = sw == A.n_sweeps - 1;
                    for (int task = warp_; task < ntask; task += NW) {
                        int tA, tB;
                        bool paired;
                        spw_task(task, e1, NT, tA, tB, paired);
                        const bool two = tB != tA;
                        const int offB = (tB - tA) * N;
                        uint32_t *SaA = S + tA * N + H;
                        const uint32_t *SoA = S + tA * N;
                        uint32_t aU0[PU], aM0[PM], aU1[PU], aM1[PM];
#pragma unroll
                        for (int k = 0; k < PU; ++k) aU0[k] = aU1[k] = 0u;
#pragma unroll
                        for (int k = 0; k < PM; ++k) aM0[k] = aM1[k] = 0u;
#pragma unroll 1
                        for (int kb = 0; kb < NB; ++kb) {
                            qq = 32 * kb + lane_;
                            if (qq < Q) {
                                uint32_t Jq[4][6];                      // (the positions are re-read per system: registers)
#pragma unroll
                                for (int e = 0; e < 4; ++e)
#pragma unroll
                                    for (int k = 0; k < 6; ++k) Jq[e][k] = JgS[(e * 6 + k) * Q + qq];
                                auto sys = [&](const int t, uint32_t *__restrict__ Sa, const uint32_t *__restrict__ So, uint32_t (&aU)[PU],
                                               uint32_t (&aM)[PM]) {
                                    const uint32_t s4[4] = {Sa[qq], Sa[Q + qq], Sa[2 * Q + qq], Sa[3 * Q + qq]};
                                    uint32_t v[4][6];
#pragma unroll
                                    for (int e = 0; e < 4; ++e)
#pragma unroll
                                        for (int k = 0; k < 6; ++k) v[e][k] = So[ixT[(e * 6 + k) * Q + qq]];
                                    const uint4 r4 = philox_rk((uint32_t)qq, time, wglob, ctr3(3, a, t), A.rk);
                                    SlotK K;
                                    {
                                        const uint4 *k4 = reinterpret_cast<const uint4 *>(thr + t * 8);
                                        const uint4 k0 = k4[0], k1 = k4[1], k2 = k4[2];
                                        K.lo[0] = k0.x; K.lo[1] = k0.y; K.lo[2] = k0.z; K.lo[3] = k0.w;
                                        K.lo[4] = k1.x; K.lo[5] = k1.y; K.lo[6] = k1.z; K.b3c = k1.w;
                                        K.nc = k2.x; K.ec = k2.y;
                                    }
                                    const uint32_t rr[4] = {r4.x, r4.y, r4.z, r4.w};
                                    uint32_t wpl[4][3], outw[4], othw[4];
#pragma unroll
                                    for (int e = 0; e < 4; ++e) {
                                        outw[e] = update_word_energy<BS>(s4[e], amask, xor3(s4[e], v[e][0], Jq[e][0]),
                                                                         xor3(s4[e], v[e][1], Jq[e][1]), xor3(s4[e], v[e][2], Jq[e][2]),
                                                                         xor3(s4[e], v[e][3], Jq[e][3]), xor3(s4[e], v[e][4], Jq[e][4]),
                                                                         xor3(s4[e], v[e][5], Jq[e][5]), rr[e], K, A.one, A.mone, wpl[e]);
                                        othw[e] = v[e][0];                     // the other colour's word at the same compact index
                                    }
                                    Sa[qq] = outw[0]; Sa[Q + qq] = outw[1]; Sa[2 * Q + qq] = outw[2]; Sa[3 * Q + qq] = outw[3];
                                    energy_accumulate(wpl, outw, othw, aU, aM);
                                };
                                sys(tA, SaA, SoA, aU0, aM0);
                                if (two) sys(tB, SaA + offB, SoA + offB, aU1, aM1);
                            }
                        }
                        spw_finish<L>(A, S, accs, aU0, aM0, aU1, aM1, tA, tB, paired, last, lane_, w, a, exchange);
                    }
                } else {
                    int bcur = -1;
                    int ix[4][6];
                    uint32_t Jq[4][6];
                    const int i0 = rank * I / NW;
                    int b = i0 / ntl, tl = i0 - b * ntl;        // tl: index among this CTA's slots
#pragma unroll 1
                    for (int i = i0; i < i1; ++i, ++tl) {
                        if (tl == ntl) { tl = 0; ++b; }
                        const int t = tlo + tl;
                        if (b != bcur) {
                            bcur = b;
                            qq = 32 * b + lane_;
                            qa = qq < Q;
                            if (!qa) qq = Q - 1;
#pragma unroll
                            for (int e = 0; e < 4; ++e) {
                                const int n = 4 * qq + e;
                                const int row = n / Lh, m = n - row * Lh;
                                const int z = row / L, y = row - z * L;
                                const int p = (colour + y + z) & 1;
                                const int sd = row * Lh + (p ? (m + 1 == Lh ? 0 : m + 1) : (m == 0 ? Lh - 1 : m - 1));
                                const int yp = (z * L + (y + 1 == L ? 0 : y + 1)) * Lh + m;
                                const int ym = (z * L + (y == 0 ? L - 1 : y - 1)) * Lh + m;
                                const int zp = ((z + 1 == L ? 0 : z + 1) * L + y) * Lh + m;
                                const int zm = ((z == 0 ? L - 1 : z - 1) * L + y) * Lh + m;
                                // slot 0: the x-neighbour at the same compact index (its bond if p, own bond else); slot 1: the one
                                // at the side index (own bond if p, its bond else)
                                constexpr auto P = G_::pos;                    // planar layout: position of a compact index
                                ix[e][0] = P(n); ix[e][1] = P(sd); ix[e][2] = P(yp); ix[e][3] = P(ym); ix[e][4] = P(zp); ix[e][5] = P(zm);
                                Jq[e][0] = p ? Joth[P(n)] : Jown[P(n)];
                                Jq[e][1] = p ? Jown[P(n)] : Joth[P(sd)];
                                Jq[e][2] = Jown[H + P(n)];      Jq[e][3] = Joth[H + P(ym)];
                                Jq[e][4] = Jown[2 * H + P(n)];  Jq[e][5] = Joth[2 * H + P(zm)];
                            }
                        }
                        uint32_t *Sa = S + tl * N + colour * H;
                        const uint32_t *So = S + tl * N + (1 - colour) * H;
                        const uint4 sv = make_uint4(Sa[qq], Sa[Q + qq], Sa[2 * Q + qq], Sa[3 * Q + qq]);   // planar: word e in array e
                        uint32_t v[4][6];
#pragma unroll
                        for (int e = 0; e < 4; ++e)
#pragma unroll
                            for (int k = 0; k < 6; ++k) v[e][k] = So[ix[e][k]];
                        const uint4 r4 = philox_rk((uint32_t)qq, time, wglob, ctr3(3, a, t), A.rk);
                        SlotK K;
                        {
                            const uint4 *k4 = reinterpret_cast<const uint4 *>(thr + t * 8);
                            const uint4 k0 = k4[0], k1 = k4[1], k2 = k4[2];
                            K.lo[0] = k0.x; K.lo[1] = k0.y; K.lo[2] = k0.z; K.lo[3] = k0.w;
                            K.lo[4] = k1.x; K.lo[5] = k1.y; K.lo[6] = k1.z; K.b3c = k1.w;
                            K.nc = k2.x; K.ec = k2.y;
                        }
                        const uint32_t s[4] = {sv.x, sv.y, sv.z, sv.w};
                        const uint32_t rr[4] = {r4.x, r4.y, r4.z, r4.w};
                        uint32_t out[4];
#pragma unroll
                        for (int e = 0; e < 4; ++e)
                            out[e] = flip_word_k<BS>(s[e], amask, xor3(s[e], v[e][0], Jq[e][0]), xor3(s[e], v[e][1], Jq[e][1]),
                                                 xor3(s[e], v[e][2], Jq[e][2]), xor3(s[e], v[e][3], Jq[e][3]),
                                                 xor3(s[e], v[e][4], Jq[e][4]), xor3(s[e], v[e][5], Jq[e][5]), rr[e], K, A.one,
                                                 A.mone);
                        if (qa) {
                            Sa[qq] = out[0]; Sa[Q + qq] = out[1]; Sa[2 * Q + qq] = out[2]; Sa[3 * Q + qq] = out[3];
                        }
                    }
                }
            }
            __syncthreads();
        }
        // ---- exchange step (R12), all in shared memory
        const bool pt_due = PT && A.pt_every > 0 && ((uint64_t)A.sweep0 + (uint64_t)sw + 1) % (uint64_t)A.pt_every == 0;
        if (pt_due && SPW) {
            exchange += 1;                                 // done by the warps of the colour-1 half sweep above
        } else if (pt_due) {
            const int lane = tid & 31, warp = tid >> 5, nwarp = nthr >> 5;
            for (int tl = warp; tl < ntl; tl += nwarp) {               // energies of the slots this CTA owns
                int U, M;
                if (A.use_tab) ladder_energy_tab<L>(S + tl * N, idxT, JgT, lane, U, M);
                else ladder_energy<L>(S + tl * N, Jsm, lane, U, M);
                Uint[(tlo + tl) * 32 + lane] = U;
                Mint[(tlo + tl) * 32 + lane] = M;
            }
            const int e1 = (int)(exchange & 1u);
            const int npairs = (NT - e1) / 2;
            // split ladder: the pair (tb, tb + 1) lies across the two CTAs of the cluster (tb = last slot of the first
            // half); it is exchanged this time iff tb has the parity of the exchange
            const int tb = (NT + 1) / 2 - 1;
            const bool cross = split_pt && tb >= e1 && ((tb - e1) & 1) == 0 && tb + 1 < NT;
            const int t_mine = half ? tb + 1 : tb, t_other = half ? tb : tb + 1;      // the cross pair's slots: mine, the partner's
            __syncthreads();
            if (cross) {
                // the partner's energies of its slot of the cross pair -> my copy of the tables (distributed shared memory)
                cluster_sync();
                if (tid < 32) {
                    Uint[t_other * 32 + tid] = (int)ld_dsmem(Uint + t_other * 32 + tid, 1 - half);
                    Mint[t_other * 32 + tid] = (int)ld_dsmem(Mint + t_other * 32 + tid, 1 - half);
                }
                __syncthreads();
            }
            const int t_end = tlo + ntl;
            for (int item = tid; item < npairs * 32; item += nthr) {       // whole warps; a cross pair is decided by both CTAs
                const int pair = item >> 5, ln = item & 31;
                const int t = e1 + 2 * pair;
                if (t + 1 < tlo || t >= t_end) continue;                   // neither slot is mine (warp-uniform)
                const int smp = w * 32 + ln;
                const int U0 = Uint[t * 32 + ln], U1 = Uint[(t + 1) * 32 + ln];
                const int M0 = Mint[t * 32 + ln], M1 = Mint[(t + 1) * 32 + ln];
                const double Et = __dsub_rn((double)(2 * U0 - 3 * N), __dmul_rn(A.h, (double)M0));
                const double Eu = __dsub_rn((double)(2 * U1 - 3 * N), __dmul_rn(A.h, (double)M1));
                const double x = __dmul_rn(__dsub_rn(A.tab[t].beta, A.tab[t + 1].beta), __dsub_rn(Et, Eu));
                const uint4 r = philox_rk(0u, (uint32_t)exchange, (uint32_t)(smp + d.s_first), ctr3(4, a, t), A.rk);
                const bool accept = (x >= 0.0) || ((uint64_t)r.x < dexp64(A.exp_tab, -x));
                const uint32_t mask = __ballot_sync(0xffffffffu, accept && smp < d.n_samples);
                if (ln == 0) {
                    masks[pair] = mask;
                    if (t >= tlo) accs[t] += (uint32_t)__popc(mask);       // counted by the CTA that owns the lower slot
                }
            }
            __syncthreads();
            if (sw == A.n_sweeps - 1) {
                for (int item = tid; item < ntl * 32; item += nthr) {      // publish the energies, permuted like the configurations
                    const int t = tlo + (item >> 5), ln = item & 31;
                    const int p = t - e1;
                    int src = t;
                    if (p >= 0 && (p >> 1) < npairs && ((masks[p >> 1] >> ln) & 1u)) src = (p & 1) ? t - 1 : t + 1;
                    const size_t o = ((size_t)(w * 32 + ln) * d.R + a) * NT + t;
                    A.U[o] = (int64_t)Uint[src * 32 + ln];
                    A.M[o] = Mint[src * 32 + ln];
                }
            }
            for (int item = tid; item < npairs * (N / 4); item += nthr) {  // masked swap of the two configurations (both mine)
                const int pair = item / (N / 4), k = item - pair * (N / 4);
                const int t = e1 + 2 * pair;
                if (t < tlo || t + 1 >= t_end) continue;
                const uint32_t mask = masks[pair];
                if (mask == 0u) continue;
                uint4 *X = reinterpret_cast<uint4 *>(S + (t - tlo) * N) + k;
                uint4 *Y = reinterpret_cast<uint4 *>(S + (t + 1 - tlo) * N) + k;
                uint4 xv = *X, yv = *Y;
                uint32_t dd;
                dd = (xv.x ^ yv.x) & mask; xv.x ^= dd; yv.x ^= dd;
                dd = (xv.y ^ yv.y) & mask; xv.y ^= dd; yv.y ^= dd;
                dd = (xv.z ^ yv.z) & mask; xv.z ^= dd; yv.z ^= dd;
                dd = (xv.w ^ yv.w) & mask; xv.w ^= dd; yv.w ^= dd;
                *X = xv;
                *Y = yv;
            }
            if (cross) {
                // the cross pair: every thread merges the partner's lanes into its words of my slot — remote reads first,
                // a cluster barrier (the partner reads MY old words meanwhile), then the local writes
                const uint32_t mask = masks[(tb - e1) >> 1];
                uint4 *X = reinterpret_cast<uint4 *>(S + (t_mine - tlo) * N);
                const uint4 *Yr = reinterpret_cast<const uint4 *>(S + (t_other - (half ? 0 : tlo + ntl)) * N);   // its local address there
                constexpr int PER = (N / 4 + Geo<L>::MAXT - 1) / Geo<L>::MAXT + 1;
                uint4 keep[PER];
                int n_keep = 0;
                if (mask != 0u)
#pragma unroll
                    for (int j = 0; j < PER; ++j) {
                        const int k = tid + j * nthr;
                        if (k < N / 4) {
                            const uint4 xv = X[k], yv = ld_dsmem4(Yr + k, 1 - half);
                            keep[j] = make_uint4(xv.x ^ ((xv.x ^ yv.x) & mask), xv.y ^ ((xv.y ^ yv.y) & mask),
                                                 xv.z ^ ((xv.z ^ yv.z) & mask), xv.w ^ ((xv.w ^ yv.w) & mask));
                            n_keep = j + 1;
                        }
                    }
                cluster_sync();
#pragma unroll
                for (int j = 0; j < PER; ++j)
                    if (j < n_keep) X[tid + j * nthr] = keep[j];
            }
            exchange += 1;
            __syncthreads();
        }
    }

    // ---- write the ladder back
    for (int t = tid; t < NT; t += nthr)
        if (accs[t]) atomicAdd(&A.pt_acc[t], (unsigned long long)accs[t]);
    {
        uint4 *dst = reinterpret_cast<uint4 *>(gOut);
        if constexpr (G_::PAIR) {
            const uint2 *src = reinterpret_cast<const uint2 *>(S);
            for (int i = tid; i < ntl * N / 4; i += nthr) {
                const int blk = i / Q, qd = i - blk * Q;
                const uint2 lo = src[blk * (2 * Q) + qd], hi = src[blk * (2 * Q) + Q + qd];
                dst[i] = make_uint4(lo.x, lo.y, hi.x, hi.y);
            }
        } else if constexpr (G_::PLANAR) {
            for (int i = tid; i < ntl * N / 4; i += nthr) {
                const int blk = i / Q, qd = i - blk * Q;
                const uint32_t *src = S + blk * H + qd;
                dst[i] = make_uint4(src[0], src[Q], src[2 * Q], src[3 * Q]);
            }
        } else {
            const uint4 *src = reinterpret_cast<const uint4 *>(S);
            for (int i = tid; i < ntl * N / 4; i += nthr) dst[i] = src[i];
        }
    }
}

// ------------------------------------------------------------------------------- host side
// nt_res slots resident in the CTA; the per-slot tables (thresholds, exchange scratch) cover all NT slots
size_t ladder_smem_bytes(int L, int NT, int nt_res)
{
    const size_t N = (size_t)L * L * L;
    return (size_t)nt_res * N * 4 + 3 * N * 4 + (size_t)NT * 8 * sizeof(uint2) + (size_t)NT * 32 * 8 + (size_t)(NT / 2 + 1) * 4 + (size_t)NT * 4;
}

// + the energy tables of ladder_energy_tab: 16 (indices) + 24 (couplings) bytes per colour-0 site, 16-byte aligned
static size_t ladder_tab_bytes(int L) { return 16 + (size_t)(L * L * L / 2) * 40; }

// A ladder that does not fit in the shared memory of one SM is split over a cluster of two CTAs (first half of the slots
// rounded up, second half); the slot pair across the two exchanges through distributed shared memory.
static bool ladder_needs_split(const Dims &d) { return ladder_smem_bytes(d.L, d.NT, d.NT) > (size_t)227 * 1024; }

bool ladder_supported(const sg_ctx *c)
{
    const Dims &d = c->d;
    if (c->path != SG_PATH_AUTO || c->kind != SG_PMJ || !d.fast_accept) return false;
    if (d.L != 4 && d.L != 6 && d.L != 8 && d.L != 10 && d.L != 12 && d.L != 16) return false;
    if (!ladder_needs_split(d)) return true;
    return d.NT >= 2 && ladder_smem_bytes(d.L, d.NT, (d.NT + 1) / 2) <= (size_t)227 * 1024;
}

template <int L>
static cudaError_t launch_l(sg_ctx *c, const LadderArgs &A, int threads, size_t smem, cudaStream_t st, int grid)
{
    constexpr bool HAS_SPW = Geo<L>::PAIR || Geo<L>::PLANAR || L == 8;
    const void *f[6] = {(const void *)k_ladder_pmj<L, false, 0>, (const void *)k_ladder_pmj<L, false, 1>,
                        (const void *)k_ladder_pmj<L, false, HAS_SPW ? 2 : 1>, (const void *)k_ladder_pmj<L, true, 0>,
                        (const void *)k_ladder_pmj<L, true, 1>, (const void *)k_ladder_pmj<L, true, HAS_SPW ? 2 : 1>};
    if (attr_needed(c, ATTR_LADDER + L / 2 - 2)) {       // L = 4..16 -> ids 1..7
        for (int i = 0; i < 6; ++i) {
            cudaError_t e = cudaFuncSetAttribute(f[i], cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
            if (e != cudaSuccess) return e;
        }
    }
    const int ptm = A.pt_every > 0 ? (A.use_spw && HAS_SPW ? 2 : 1) : 0;
    const void *kern = f[(A.d.bs_accept ? 3 : 0) + ptm];
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3((unsigned)threads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    if (ptm != 0 && A.split) {
        // split ladders with exchanges: the two CTAs of a ladder are a thread-block cluster (distributed shared memory)
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = 2;
        at[0].val.clusterDim.y = 1;
        at[0].val.clusterDim.z = 1;
        cfg.attrs = at;
        cfg.numAttrs = 1;
    }
    void *args[1] = {(void *)&A};
    return cudaLaunchKernelExC(&cfg, kern, args);
}

// n_sweeps consecutive sweeps starting at global sweep index `sweep0`, with the exchanges that fall due fused in
// (pt_every > 0; first exchange index exchange0); returns kernels launched (or -1)
int launch_ladder_pmj(sg_ctx *c, uint64_t sweep0, int n_sweeps, uint64_t exchange0, int pt_every, uint32_t *spins_out)
{
    const Dims &d = c->d;
    LadderArgs A;
    A.d = d;
    A.spins = c->spins;
    A.spins_out = spins_out ? spins_out : c->spins;
    A.J = c->J;
    A.tab = c->tab;
    for (int r = 0; r < 10; ++r) {
        A.rk[2 * r] = d.k0 + (uint32_t)r * 0x9E3779B9u;
        A.rk[2 * r + 1] = d.k1 + (uint32_t)r * 0xBB67AE85u;
    }
    A.pad0 = 0;
    A.sweep0 = (uint32_t)sweep0;
    A.n_sweeps = n_sweeps;
    A.pt_every = pt_every;
    A.exchange0 = exchange0;
    A.exp_tab = c->exp64_tab;
    A.h = c->h;
    A.one = 1u;
    A.mone = 0xffffffffu;
    A.U = c->U;
    A.M = c->M;
    A.pt_acc = c->pt_acc;
    const int Q = d.N / 8;
    A.split = ladder_needs_split(d) ? 1 : 0;
    A.nt_res = A.split ? (d.NT + 1) / 2 : d.NT;
    // groups: as many as fit in <= 512 threads, at most the resident slots, preferring a divisor of their number
    const int maxt = (d.L / 2) % 4 == 0 ? 512 : 384;
    int G = std::max(1, std::min(A.nt_res, maxt / Q));
    for (int gtry = G; gtry >= 1 && gtry * 2 > G; --gtry)
        if (A.nt_res % gtry == 0) { G = gtry; break; }
    A.G = G;
    int threads = (Q * G + 31) / 32 * 32;
    if ((d.L / 2) % 4 != 0) {
        // generic lattices: balanced warp items (block of 32 quads, system); a multiple of four warps, at most 12
        const int items = (Q + 31) / 32 * A.nt_res;
        // (measured at C3: 12 warps with 130 registers beat 16 with 116 and 20 with 96 - the kernel is bound by ALU-pipe
        // and issue throughput, not by latency)
        threads = 32 * std::min(12, (items + 3) / 4 * 4);
    }
    if (threads > maxt) return -1;
    if (A.split && ((d.N / 4 + maxt - 1) / maxt + 1) * threads < d.N / 4) return -1;   // (cross-pair swap: PER quads per thread)
    size_t smem = ladder_smem_bytes(d.L, d.NT, A.nt_res);
    const bool pair = (d.L / 2) % 4 != 0 && (d.L / 2) % 2 == 0;                 // Geo<L>::PAIR
    const bool planar = (d.L / 2) % 2 == 1;                                     // Geo<L>::PLANAR
    // tables of the warp-per-pair exchange half sweep: 9 offset pairs per quad (pair layout), 24 positions + 24 coupling
    // words per quad (planar layout)
    const size_t spw_bytes = 16 + (size_t)Q * (pair ? 72 : 192);
    A.use_spw = (pair || planar) && !A.split && smem + spw_bytes <= (size_t)227 * 1024 ? 1 : 0;
    if (d.L == 8 && !A.split) A.use_spw = 1;                                    // rows of whole quads: no table needed
    A.use_tab = !A.use_spw && smem + ladder_tab_bytes(d.L) <= (size_t)227 * 1024 ? 1 : 0;
    if (A.use_spw && (pair || planar)) smem += spw_bytes;
    if (A.use_tab) smem += ladder_tab_bytes(d.L);
    int grid = d.W * d.R;
    A.n_full = grid;
    if (A.split) {
        A.n_full = 0;
        grid *= 2;
    } else if (pt_every == 0 && d.NT >= 2) {
        // plain sweeps, one CTA per SM: if the last wave of ladders fills at most half of the SMs, each of its ladders
        // goes to two CTAs (C3: 512 ladders on 148 SMs = 3 waves + 68 -> 136 half ladders: 3.5 instead of 4 wave times)
        int dev = 0, n_sm = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
        const int slots = smem > (size_t)113 * 1024 ? n_sm : 0;                // only where one CTA fills an SM
        const int tail = slots > 0 ? grid % slots : 0;
        if (slots > 0 && grid > slots && tail > 0 && 2 * tail <= slots) {
            A.n_full = grid - tail;
            grid = A.n_full + 2 * tail;
        }
    }
    cudaError_t e;
    switch (d.L) {
    case 4: e = launch_l<4>(c, A, threads, smem, c->stream, grid); break;
    case 6: e = launch_l<6>(c, A, threads, smem, c->stream, grid); break;
    case 8: e = launch_l<8>(c, A, threads, smem, c->stream, grid); break;
    case 10: e = launch_l<10>(c, A, threads, smem, c->stream, grid); break;
    case 12: e = launch_l<12>(c, A, threads, smem, c->stream, grid); break;
    case 16: e = launch_l<16>(c, A, threads, smem, c->stream, grid); break;
    default: return -1;
    }
    return e == cudaSuccess ? 1 : -1;
}

}  // namespace sg
