// sg_tpack.cu — the paper's own packing ("Multispin coding is used to pack the N_T replicas into the
// small but extremely fast shared memory"; R17), coupling_kind = SG_PMJ_TPACK.
//
// One 32-bit word per lattice site holds the spins of the temperature copies of ONE (sample, replica): bit tl of
// word j is slot t = 32 j + tl (N_T <= 64: one or two words per site).  The couplings are common to all bits
// (6 bits per site, expanded to 0 / ~0 words on the fly), the lattice of a (sample, replica) lives in the shared
// memory of one CTA for all sweeps of a launch, and parallel tempering is a bit permutation inside the word
// (masked delta swap of neighbouring bits; one extra swap across the word boundary for N_T > 32).
//
// R17: every temperature copy keeps its OWN 32-bit Philox draw per site (the draws of slot t are exactly those of
// the sample-packed layout, R5/R6), because sharing one draw among the temperature bits of a word — the cheap
// multispin trick that is valid for independent samples — correlates the chains that parallel tempering swaps and
// biases the Boltzmann averages (measured on the 2x2x2 enumeration pin: <E> off by 44 sigma at the hottest slot).
// The trajectory of a sample is therefore bit-identical to the one of SG_PMJ, and the same oracle checks it; what
// differs is the cost profile: one Philox call per (slot, quad) and a per-bit threshold compare, ~22 instructions
// per flip attempt instead of ~2, in exchange for full lanes when there are few samples but many temperatures.
//
// Everything outside the sweep + exchange loop (initial state, overlaps, energies for the getters, read-back) runs
// on the sample-packed copy of the state; k_tp_from_std / k_tp_to_std convert between the two layouts with one
// 32 x 32 warp bit-transpose per site (rows = slots, columns = samples of a packed word).
#include "sg_device.cuh"
#include "sg_accept.cuh"
#include "sg_internal.h"

namespace sg {

struct TpArgs {
    Dims d;
    uint32_t *tps;            // [S][R][NW][2][H]  bit tl of word j = slot 32 j + tl
    const uint8_t *J6;        // [S][2][H]  bit k: bond to neighbour k (+x, -x, +y, -y, +z, -z) is J = -1
    const SlotTab *tab;
    const double *exp_tab;
    double h;
    uint32_t rk[20];
    uint64_t sweep0, exchange0;
    int n_sweeps, pt_every;
    int NW;                   // words per site: ceil(NT / 32)
    int wpb;                  // unused (one CTA per lattice)
    int64_t *U;               // [S][R][NT] the kernel's own energies after the last exchange of the launch
    int32_t *M;
    unsigned long long *pt_acc;
};

namespace {

// neighbour compact indices (in the other colour's array) of element n of colour c, compile-time L
template <int L>
__device__ __forceinline__ void nbr6(int c, int n, int (&ix)[6])
{
    constexpr int Lh = L / 2;
    const int row = n / Lh, m = n - row * Lh;
    const int z = row / L, y = row - z * L;
    const int p = (c + y + z) & 1;
    const int sd = row * Lh + (p ? (m + 1 == Lh ? 0 : m + 1) : (m == 0 ? Lh - 1 : m - 1));
    ix[0] = p ? sd : n;                                                  // +x
    ix[1] = p ? n : sd;                                                  // -x
    ix[2] = (z * L + (y + 1 == L ? 0 : y + 1)) * Lh + m;                 // +y
    ix[3] = (z * L + (y == 0 ? L - 1 : y - 1)) * Lh + m;                 // -y
    ix[4] = ((z + 1 == L ? 0 : z + 1) * L + y) * Lh + m;                 // +z
    ix[5] = ((z == 0 ? L - 1 : z - 1) * L + y) * Lh + m;                 // -z
}

constexpr int TP_THREADS = 256;

// One CTA per (sample, replica) lattice.  Work item of a half sweep = (quad q, word j, group of 8 slots): the thread
// counts the unsatisfied bonds of the quad's 4 sites for all slots of the word (bitwise, so the other groups' bits cost
// nothing), then draws and decides its 8 slots and flips them with one atomicXor per site word (the groups of a word
// touch disjoint bits, and no thread reads bits of another group).
// SPI = slots per item: 8 when there are few lattices (more threads per lattice, lower latency), 32 when the GPU is
// full anyway (the bond counting and the neighbour indices of a quad are then shared by all slots of the word).
template <int L, int SPI>
__global__ void __launch_bounds__(TP_THREADS) k_tp_run(const __grid_constant__ TpArgs A)
{
    constexpr int N = L * L * L, H = N / 2, Q = H / 4;
    extern __shared__ __align__(16) unsigned char sm_raw[];
    const Dims &d = A.d;
    const int NT = d.NT, NW = A.NW;
    uint2 *thr = reinterpret_cast<uint2 *>(sm_raw);                      // [NT][7][2] thresholds as (lo, hi) of thr in [0, 2^32]
    uint32_t *spread = reinterpret_cast<uint32_t *>(thr + NT * 14);      // [256] bit i of the index -> bit 4 i
    uint32_t *S = spread + 256;                                          // [NW][2][H]
    int *UM = reinterpret_cast<int *>(S + (size_t)NW * N);               // [2 (U, M)][NW][32] per-slot energies
    uint32_t *masks = reinterpret_cast<uint32_t *>(UM + 4 * 32);         // [NW] accepted lower slots of the exchange
    uint8_t *Jb = reinterpret_cast<uint8_t *>(masks + 4);                // [2][H]
    const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5;

    for (int i = tid; i < NT * 14; i += nthr) {
        const uint2 v = A.tab[i / 14].c64g[(i % 14) >> 1][i & 1];        // (uint64)(0 - thr)
        const uint64_t th = (uint64_t)0 - (((uint64_t)v.y << 32) | v.x);
        thr[i] = make_uint2((uint32_t)th, (uint32_t)(th >> 32));
    }
    for (int i = tid; i < 256; i += nthr) {
        uint32_t x = 0;
        for (int b = 0; b < 8; ++b) x |= ((uint32_t)(i >> b) & 1u) << (4 * b);
        spread[i] = x;
    }
    const int lat = blockIdx.x;                                          // (sample, replica) lattice of this CTA
    const int s = lat / d.R, a = lat % d.R;
    uint32_t *gS = A.tps + (size_t)lat * NW * N;
    for (int i = tid; i < NW * N / 4; i += nthr) reinterpret_cast<uint4 *>(S)[i] = reinterpret_cast<const uint4 *>(gS)[i];
    {
        const uint32_t *gJ = reinterpret_cast<const uint32_t *>(A.J6 + (size_t)s * N);
        for (int i = tid; i < N / 4; i += nthr) reinterpret_cast<uint32_t *>(Jb)[i] = gJ[i];
    }
    __syncthreads();

    const uint32_t amask = d.neg_h ? 0xffffffffu : 0u;
    const uint32_t wglob = (uint32_t)((s + d.s_first) >> 5);             // sweep draws are keyed by the packed word of the sample (R5)
    const uint32_t sglob = (uint32_t)(s + d.s_first);
    uint64_t exchange = A.exchange0;
    uint32_t cnt[2] = {0u, 0u};                                          // warp 0: accepted swaps with this lane's slot as the lower one
    constexpr int NG = 32 / SPI;                                         // slot groups (items) per word
    const int n_items = Q * NW * NG;

    for (int sw = 0; sw < A.n_sweeps; ++sw) {
        const uint64_t sweep = A.sweep0 + (uint64_t)sw;
#pragma unroll 1
        for (int colour = 0; colour < 2; ++colour) {
            const uint32_t time = 2u * (uint32_t)sweep + (uint32_t)colour;
#pragma unroll 1
            for (int item = tid; item < n_items; item += nthr) {
                const int q = item % Q, rest = item / Q;                 // consecutive threads: consecutive quads (conflict-free)
                const int j = rest % NW, tb0 = SPI * (rest / NW);
                const int nb = NT - 32 * j < 32 ? NT - 32 * j : 32;      // slots in this word
                if (tb0 >= nb) continue;
                uint32_t *Sa = S + (size_t)j * N + colour * H;
                const uint32_t *So = S + (size_t)j * N + (1 - colour) * H;
                const uint32_t jq = reinterpret_cast<const uint32_t *>(Jb + colour * H)[q];
                uint32_t al[4], n0[4], n1[4], n2[4];                     // field alignment and unsatisfied-bond count planes
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    int ix[6];
                    nbr6<L>(colour, 4 * q + e, ix);
                    const uint32_t j6 = (jq >> (8 * e)) & 0xffu;
                    const uint32_t sp = Sa[4 * q + e];
                    uint32_t u[6];
#pragma unroll
                    for (int k = 0; k < 6; ++k) u[k] = xor3(sp, So[ix[k]], 0u - ((j6 >> k) & 1u));
                    const uint32_t s0 = xor3(u[0], u[1], u[2]), c0 = maj3(u[0], u[1], u[2]);
                    const uint32_t s1 = xor3(u[3], u[4], u[5]), c1 = maj3(u[3], u[4], u[5]);
                    const uint32_t kk = s0 & s1;
                    n0[e] = s0 ^ s1;
                    n1[e] = xor3(c0, c1, kk);
                    n2[e] = maj3(c0, c1, kk);
                    al[e] = sp ^ amask;
                }
#pragma unroll 1
              for (int tb = tb0; tb < tb0 + SPI && tb < nb; tb += 8) {
                uint32_t cw[4];                                          // class nibbles of 8 slots: a | n0 << 1 | n1 << 2 | n2 << 3 = a + 2 n_u
#pragma unroll
                for (int e = 0; e < 4; ++e)
                    cw[e] = spread[(al[e] >> tb) & 0xffu] | (spread[(n0[e] >> tb) & 0xffu] << 1) |
                            (spread[(n1[e] >> tb) & 0xffu] << 2) | (spread[(n2[e] >> tb) & 0xffu] << 3);
                uint32_t acc[4] = {0u, 0u, 0u, 0u};
#pragma unroll
                for (int t8 = 0; t8 < 8; ++t8) {
                    const int tl = tb + t8;
                    if (tl < nb) {
                        const int t = 32 * j + tl;
                        const uint4 r4 = philox_rk8((uint32_t)q, time, wglob, ctr3(3, a, t), A.rk);
                        const uint32_t rr[4] = {r4.x, r4.y, r4.z, r4.w};
                        const uint2 *tt = thr + t * 14;
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            const uint2 th = tt[(cw[e] >> (4 * t8)) & 15u];      // nibble = a + 2 n_u = index into thr[t][n_u][a]
                            const bool flip = th.y != 0u || rr[e] < th.x;         // (uint64) r < thr
                            acc[e] |= flip ? (1u << t8) : 0u;
                        }
                    }
                }
#pragma unroll
                for (int e = 0; e < 4; ++e)
                    if (acc[e]) atomicXor(&Sa[4 * q + e], acc[e] << tb);
              }
            }
            __syncthreads();
        }
        // ---- exchange step (R12): per-bit energies, decisions by the lane of the lower slot (warp 0), bit permutation
        if (A.pt_every > 0 && (sweep + 1) % (uint64_t)A.pt_every == 0) {
            if (tid < 4 * 32) UM[tid] = 0;
            __syncthreads();
            for (int j = 0; j < NW; ++j) {
                const uint32_t *s0 = S + (size_t)j * N, *s1 = s0 + H;
                uint32_t bigU[10], bigM[8], inU[7], inM[6];              // per thread: <= ceil(H / 256) = 8 sites -> U <= 48, M <= 16
#pragma unroll
                for (int k = 0; k < 10; ++k) bigU[k] = 0;
#pragma unroll
                for (int k = 0; k < 8; ++k) bigM[k] = 0;
#pragma unroll
                for (int k = 0; k < 7; ++k) inU[k] = 0;
#pragma unroll
                for (int k = 0; k < 6; ++k) inM[k] = 0;
                int pending = 0;
                for (int n = tid; n < H; n += nthr) {                    // the six bonds of every colour-0 site cover each bond once
                    int ix[6];
                    nbr6<L>(0, n, ix);
                    const uint32_t sa = s0[n], sb = s1[n], jb = Jb[n];
                    uint32_t u[6];
#pragma unroll
                    for (int k = 0; k < 6; ++k) u[k] = xor3(sa, s1[ix[k]], 0u - ((jb >> k) & 1u));
                    const uint32_t a0 = xor3(u[0], u[1], u[2]), c0 = maj3(u[0], u[1], u[2]);
                    const uint32_t a1 = xor3(u[3], u[4], u[5]), c1 = maj3(u[3], u[4], u[5]);
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
                atomicAdd(&UM[j * 32 + lane], (int)bs_warp_total(bigU, 10, lane));
                atomicAdd(&UM[64 + j * 32 + lane], (int)bs_warp_total(bigM, 8, lane));
            }
            __syncthreads();
            const int e1 = (int)(exchange & 1u);
            if (warp == 0) {
                int Ureg[2], Mreg[2];
                uint32_t mask[2] = {0u, 0u};
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    Ureg[j] = j < NW ? UM[j * 32 + lane] : 0;
                    Mreg[j] = j < NW ? 2 * UM[64 + j * 32 + lane] - N : 0;
                }
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    if (j >= NW) continue;
                    const int t = 32 * j + lane;
                    // partner = slot t + 1: the next lane, or lane 0 of the next word
                    int Up = __shfl_down_sync(0xffffffffu, Ureg[j], 1), Mp = __shfl_down_sync(0xffffffffu, Mreg[j], 1);
                    if (j == 0) {
                        const int U0 = __shfl_sync(0xffffffffu, Ureg[1], 0), M0 = __shfl_sync(0xffffffffu, Mreg[1], 0);
                        if (lane == 31) { Up = U0; Mp = M0; }
                    }
                    bool accept = false;
                    if ((t & 1) == e1 && t + 1 < NT) {
                        const double Et = __dsub_rn((double)(2 * Ureg[j] - 3 * N), __dmul_rn(A.h, (double)Mreg[j]));
                        const double Eu = __dsub_rn((double)(2 * Up - 3 * N), __dmul_rn(A.h, (double)Mp));
                        const double x = __dmul_rn(__dsub_rn(A.tab[t].beta, A.tab[t + 1].beta), __dsub_rn(Et, Eu));
                        const uint4 r = philox_rk8(0u, (uint32_t)exchange, sglob, ctr3(4, a, t), A.rk);
                        accept = (x >= 0.0) || ((uint64_t)r.x < dexp64(A.exp_tab, -x));
                    }
                    mask[j] = __ballot_sync(0xffffffffu, accept);
                    cnt[j] += accept ? 1u : 0u;
                }
                if (lane < 2) masks[lane] = mask[lane];
                if (sw == A.n_sweeps - 1) {                              // publish the kernel's own energies, permuted like the configurations
#pragma unroll
                    for (int j = 0; j < 2; ++j) {
                        if (j >= NW) continue;
                        const int Ud = __shfl_down_sync(0xffffffffu, Ureg[j], 1), Md = __shfl_down_sync(0xffffffffu, Mreg[j], 1);
                        const int Uu = __shfl_up_sync(0xffffffffu, Ureg[j], 1), Mu = __shfl_up_sync(0xffffffffu, Mreg[j], 1);
                        const int Ux = __shfl_sync(0xffffffffu, Ureg[j ^ 1], j == 0 ? 0 : 31), Mx = __shfl_sync(0xffffffffu, Mreg[j ^ 1], j == 0 ? 0 : 31);
                        int Un = Ureg[j], Mn = Mreg[j];
                        if (lane < 31 && ((mask[j] >> lane) & 1u)) { Un = Ud; Mn = Md; }
                        if (lane > 0 && ((mask[j] >> (lane - 1)) & 1u)) { Un = Uu; Mn = Mu; }
                        if (NW == 2 && (mask[0] >> 31) && ((j == 0 && lane == 31) || (j == 1 && lane == 0))) { Un = Ux; Mn = Mx; }
                        const int t = 32 * j + lane;
                        if (t < NT) {
                            const size_t o = ((size_t)s * d.R + a) * NT + t;
                            A.U[o] = (int64_t)Un;
                            A.M[o] = Mn;
                        }
                    }
                }
            }
            __syncthreads();
            // bit permutation of every site word: swap bits (tl, tl + 1) for the accepted lower slots tl
            for (int j = 0; j < NW; ++j) {
                const uint32_t m = masks[j] & 0x7fffffffu;
                if (m == 0u) continue;                                   // block-uniform
                uint32_t *Sj = S + (size_t)j * N;
                for (int n = tid; n < N; n += nthr) {
                    const uint32_t x = Sj[n];
                    const uint32_t tt = ((x >> 1) ^ x) & m;
                    Sj[n] = x ^ tt ^ (tt << 1);
                }
            }
            if (NW == 2 && (masks[0] >> 31)) {                           // pair (31, 32): bit 31 of word 0 <-> bit 0 of word 1
                for (int n = tid; n < N; n += nthr) {
                    const uint32_t x = S[n], y = S[N + n];
                    const uint32_t dd = ((x >> 31) ^ y) & 1u;
                    S[n] = x ^ (dd << 31);
                    S[N + n] = y ^ dd;
                }
            }
            exchange += 1;
            __syncthreads();
        }
    }
    if (warp == 0) {
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            const int t = 32 * j + lane;
            if (j < NW && t < NT && cnt[j]) atomicAdd(&A.pt_acc[t], (unsigned long long)cnt[j]);
        }
    }
    for (int i = tid; i < NW * N / 4; i += nthr) reinterpret_cast<uint4 *>(gS)[i] = reinterpret_cast<const uint4 *>(S)[i];
}

// ------------------------------------------------------------------------ layout conversion
// sample-packed: std[w][a][t][c][n], bit l = sample 32 w + l;  temperature-packed: tps[s][a][j][c][n], bit tl = slot 32 j + tl.
// One warp per (w, a, j): for every site, lane tl loads the word of slot 32 j + tl (row tl), the warp transposes the
// 32 x 32 bit matrix, lane l stores the word of sample 32 w + l.
__global__ void __launch_bounds__(128)
k_tp_from_std(Dims d, int NW, const uint32_t *__restrict__ stdw, uint32_t *__restrict__ tps)
{
    const int lane = threadIdx.x & 31;
    const long long g = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (g >= (long long)d.W * d.R * NW) return;
    const int j = (int)(g % NW), a = (int)((g / NW) % d.R), w = (int)(g / ((long long)NW * d.R));
    const int t = 32 * j + lane, smp = 32 * w + lane;
    const uint32_t *src = stdw + (((size_t)w * d.R + a) * d.NT + (t < d.NT ? t : 0)) * d.N;
    uint32_t *dst = tps + (((size_t)(smp < d.n_samples ? smp : 0) * d.R + a) * NW + j) * d.N;
    for (int n = 0; n < d.N; ++n) {
        const uint32_t row = t < d.NT ? src[n] : 0u;
        const uint32_t col = transpose32(row, lane);
        if (smp < d.n_samples) dst[n] = col;
    }
}

__global__ void __launch_bounds__(128)
k_tp_to_std(Dims d, int NW, const uint32_t *__restrict__ tps, uint32_t *__restrict__ stdw)
{
    const int lane = threadIdx.x & 31;
    const long long g = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (g >= (long long)d.W * d.R * NW) return;
    const int j = (int)(g % NW), a = (int)((g / NW) % d.R), w = (int)(g / ((long long)NW * d.R));
    const int t = 32 * j + lane, smp = 32 * w + lane;
    const uint32_t *src = tps + (((size_t)(smp < d.n_samples ? smp : 0) * d.R + a) * NW + j) * d.N;
    uint32_t *dst = stdw + (((size_t)w * d.R + a) * d.NT + (t < d.NT ? t : 0)) * d.N;
    for (int n = 0; n < d.N; ++n) {
        const uint32_t row = smp < d.n_samples ? src[n] : 0u;         // row = sample, bits = slots
        const uint32_t col = transpose32(row, lane);                    // lane tl: bits = samples
        if (t < d.NT) dst[n] = col;
    }
}

// J6[s][c][n]: the six bond bits of site (c, n) of sample s from the sample-packed couplings J[w][c][dir][n]
__global__ void __launch_bounds__(256)
k_tp_pack_J(Dims d, const uint32_t *__restrict__ J, uint8_t *__restrict__ J6)
{
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= (long long)d.n_samples * d.N) return;
    const int k = (int)(tid % d.N), s = (int)(tid / d.N);
    const int c = k / d.H, n = k - c * d.H;
    const int w = s >> 5, l = s & 31;
    const int H = d.H, L = d.L, Lh = d.Lh;
    const int row = n / Lh, m = n - row * Lh;
    const int z = row / L, y = row - z * L;
    const int p = (c + y + z) & 1;
    const int sd = row * Lh + (p ? (m + 1 == Lh ? 0 : m + 1) : (m == 0 ? Lh - 1 : m - 1));
    const int xm = p ? n : sd;
    const int ym = (z * L + (y == 0 ? L - 1 : y - 1)) * Lh + m;
    const int zm = ((z == 0 ? L - 1 : z - 1) * L + y) * Lh + m;
    const uint32_t *Jown = J + ((size_t)(w * 2 + c) * 3) * H;
    const uint32_t *Joth = J + ((size_t)(w * 2 + 1 - c) * 3) * H;
    uint32_t b = 0;
    b |= ((Jown[n] >> l) & 1u) << 0;
    b |= ((Joth[xm] >> l) & 1u) << 1;
    b |= ((Jown[H + n] >> l) & 1u) << 2;
    b |= ((Joth[H + ym] >> l) & 1u) << 3;
    b |= ((Jown[2 * H + n] >> l) & 1u) << 4;
    b |= ((Joth[2 * H + zm] >> l) & 1u) << 5;
    J6[tid] = (uint8_t)b;
}

size_t tp_smem(int L, int NT)
{
    const size_t N = (size_t)L * L * L;
    const int NW = (NT + 31) / 32;
    return (size_t)NT * 14 * 8 + 1024 + (size_t)NW * N * 4 + 4 * 32 * 4 + 16 + N;
}

template <int L>
cudaError_t launch_tp(sg_ctx *c, const TpArgs &A, size_t smem, int grid)
{
    if (attr_needed(c, ATTR_TPACK + L / 2 - 2)) {        // L = 4..16 -> ids 24..30
        cudaError_t e = cudaFuncSetAttribute(k_tp_run<L, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(k_tp_run<L, 32>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
        if (e != cudaSuccess) return e;
    }
    int dev = 0, n_sm = 0;
    cudaGetDevice(&dev);
    if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n_sm <= 0) n_sm = 148;
    if (grid >= n_sm * 6) k_tp_run<L, 32><<<grid, TP_THREADS, smem, c->stream>>>(A);     // enough lattices to fill every SM
    else k_tp_run<L, 8><<<grid, TP_THREADS, smem, c->stream>>>(A);
    return cudaGetLastError();
}

}  // namespace

size_t tp_state_bytes(int L, int n_samples, int R, int NT) { return (size_t)n_samples * R * ((NT + 31) / 32) * L * L * L * 4; }

bool tp_supported(const sg_ctx *c)
{
    const Dims &d = c->d;
    if (c->kind != SG_PMJ_TPACK || c->path != SG_PATH_AUTO) return false;
    if (d.L != 4 && d.L != 6 && d.L != 8 && d.L != 10 && d.L != 12 && d.L != 16) return false;
    return tp_smem(d.L, d.NT) <= (size_t)227 * 1024;
}

int launch_tp_pack_J(sg_ctx *c)
{
    const Dims &d = c->d;
    const long long n = (long long)d.n_samples * d.N;
    k_tp_pack_J<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(d, c->J, c->J6);
    return 1;
}

int launch_tp_from_std(sg_ctx *c)
{
    const Dims &d = c->d;
    const int NW = (d.NT + 31) / 32;
    const long long n = (long long)d.W * d.R * NW;
    k_tp_from_std<<<(unsigned)((n + 3) / 4), 128, 0, c->stream>>>(d, NW, c->spins, c->tps);
    return 1;
}

int launch_tp_to_std(sg_ctx *c)
{
    const Dims &d = c->d;
    const int NW = (d.NT + 31) / 32;
    const long long n = (long long)d.W * d.R * NW;
    k_tp_to_std<<<(unsigned)((n + 3) / 4), 128, 0, c->stream>>>(d, NW, c->tps, c->spins);
    return 1;
}

// n_sweeps sweeps on the temperature-packed state with the exchanges that fall due fused in; 1 launch or -1
int launch_tp_run(sg_ctx *c, uint64_t sweep0, int n_sweeps, uint64_t exchange0, int pt_every)
{
    const Dims &d = c->d;
    TpArgs A;
    A.d = d;
    A.tps = c->tps;
    A.J6 = c->J6;
    A.tab = c->tab;
    A.exp_tab = c->exp64_tab;
    A.h = c->h;
    for (int r = 0; r < 10; ++r) {
        A.rk[2 * r] = d.k0 + (uint32_t)r * 0x9E3779B9u;
        A.rk[2 * r + 1] = d.k1 + (uint32_t)r * 0xBB67AE85u;
    }
    A.sweep0 = sweep0;
    A.exchange0 = exchange0;
    A.n_sweeps = n_sweeps;
    A.pt_every = pt_every;
    A.NW = (d.NT + 31) / 32;
    A.wpb = 1;
    A.U = c->U;
    A.M = c->M;
    A.pt_acc = c->pt_acc;
    const size_t smem = tp_smem(d.L, d.NT);
    const int grid = d.n_samples * d.R;
    cudaError_t e;
    switch (d.L) {
    case 4: e = launch_tp<4>(c, A, smem, grid); break;
    case 6: e = launch_tp<6>(c, A, smem, grid); break;
    case 8: e = launch_tp<8>(c, A, smem, grid); break;
    case 10: e = launch_tp<10>(c, A, smem, grid); break;
    case 12: e = launch_tp<12>(c, A, smem, grid); break;
    case 16: e = launch_tp<16>(c, A, smem, grid); break;
    default: return -1;
    }
    return e == cudaSuccess ? 1 : -1;
}

}  // namespace sg
