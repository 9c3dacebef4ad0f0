// sg_ladder8.cu — L = 8 specialisation of the shared-memory ladder kernel (BASELINE.json config 2),
// with parallel tempering fused in: one launch runs `n_sweeps` sweeps and every exchange that falls
// due between them, without leaving the SM.
//
// L = 8: a quad (4 same-colour sites = one Philox call) is exactly one (y, z) row.  Rows are kept in
// shared memory sorted by the parity pi = (y+z)&1 ("slot" order), so that every warp owns 32 rows of
// one parity: the row parity p = (colour + pi) & 1 that decides whether the second x-neighbour sits
// at m-1 or m+1 is then warp-uniform and becomes a static register renaming (no selects, no extra
// loads, no bank conflicts: all neighbour rows of a quarter-warp are contiguous 128-byte runs).
// Thread (g, pi, j) owns slot pi*32+j for the systems t = g, g+G, ...; the two warps of a group only
// synchronise with each other (named barrier) between half sweeps.
//
// Exchange step (R12), all in shared memory: per-lane U and M of every system are reduced from the
// bit planes produced during the colour-1 half sweep (U = sum over colour-1 sites of their post-flip
// unsatisfied count; M = sum of all spin words) by three bit-sliced 4:1 adder stages and one warp
// bit-transpose per system; one thread per (pair, lane) decides; masked swap of the two systems.
#include "sg_accept.cuh"
#include "sg_device.cuh"
#include "sg_internal.h"

namespace sg {

struct Ladder8Args {
    Dims d;
    uint32_t *spins;          // state the launch starts from
    uint32_t *spins_out;      // where it leaves the state (the same buffer, or the second one: see sg_run)
    const uint32_t *J;
    const SlotTab *tab;
    const double *exp_tab;
    double h;
    uint32_t rk[20];
    uint64_t sweep0;          // global index of the first sweep of this launch
    uint64_t exchange0;       // global index of the first exchange of this launch
    int n_sweeps;
    int pt_every;             // 0 = never
    int G;
    uint32_t one, mone;       // 1 and 0xFFFFFFFF as run-time values: mad.lo with them stays an IMAD (FMA pipe)
    int64_t *U;               // [32 W][R][NT]: the kernel's own per-lane energies after the LAST exchange of the launch
    int32_t *M;               //                (post-swap), written only if that exchange follows the last sweep
    unsigned long long *pt_acc;   // [NT] accepted swaps per lower slot of the pair
};

__device__ __forceinline__ int slot_of_row(int y, int z) { return ((y + z) & 1) * 32 + z * 4 + (y >> 1); }

constexpr int PU1 = 5, PM1 = 4;             // planes per thread after the in-thread stage (U <= 24, M <= 8)
constexpr int PW1 = PU1 + PM1;              // words per (system, thread) in the reduction buffer

// 4:1 adder stage over the reduction buffer: in[sys][PU+PM][n_in] -> out[sys][PU+2+PM+2][n_in/4]
template <int PU, int PM>
__device__ __forceinline__ void reduce4_item(const uint32_t *__restrict__ in, uint32_t *__restrict__ out, int sys, int n_in, int c)
{
    const int n_out = n_in >> 2;
    {
        const uint32_t *src = in + (size_t)sys * (PU + PM) * n_in + 4 * c;
        uint32_t a[PU], b[PU], ab[PU + 1], cd[PU + 1], u[PU + 2];
#pragma unroll
        for (int k = 0; k < PU; ++k) { a[k] = src[k * n_in]; b[k] = src[k * n_in + 1]; }
        bs_sum<PU>(a, b, ab);
#pragma unroll
        for (int k = 0; k < PU; ++k) { a[k] = src[k * n_in + 2]; b[k] = src[k * n_in + 3]; }
        bs_sum<PU>(a, b, cd);
        bs_sum<PU + 1>(ab, cd, u);
        uint32_t ma[PM], mb[PM], mab[PM + 1], mcd[PM + 1], m[PM + 2];
        const uint32_t *srm = src + PU * n_in;
#pragma unroll
        for (int k = 0; k < PM; ++k) { ma[k] = srm[k * n_in]; mb[k] = srm[k * n_in + 1]; }
        bs_sum<PM>(ma, mb, mab);
#pragma unroll
        for (int k = 0; k < PM; ++k) { ma[k] = srm[k * n_in + 2]; mb[k] = srm[k * n_in + 3]; }
        bs_sum<PM>(ma, mb, mcd);
        bs_sum<PM + 1>(mab, mcd, m);
        uint32_t *dst = out + (size_t)sys * (PU + PM + 4) * n_out + c;
#pragma unroll
        for (int k = 0; k < PU + 2; ++k) dst[k * n_out] = u[k];
#pragma unroll
        for (int k = 0; k < PM + 2; ++k) dst[(PU + 2 + k) * n_out] = m[k];
    }
}

template <int PU, int PM>
__device__ __forceinline__ void reduce4(const uint32_t *__restrict__ in, uint32_t *__restrict__ out, int n_sys,
                                        int n_in, int tid, int nthr)
{
    const int n_out = n_in >> 2;
    for (int item = tid; item < n_sys * n_out; item += nthr) reduce4_item<PU, PM>(in, out, item / n_out, n_in, item % n_out);
}

template <int P, bool ENERGY, bool BS>
__device__ __forceinline__ void half_sweep_quad(uint32_t *__restrict__ Sa, const uint32_t *__restrict__ So, int slot,
                                                int s_yp, int s_ym, int s_zp, int s_zm, const uint32_t (&JA)[4],
                                                const uint32_t (&JB)[4], const uint32_t (&Jyp)[4],
                                                const uint32_t (&Jym)[4], const uint32_t (&Jzp)[4],
                                                const uint32_t (&Jzm)[4], const uint4 r4, const uint4 *__restrict__ thr_t,
                                                uint32_t amask, uint32_t one, uint32_t mone, uint32_t *__restrict__ red)
{
    const uint4 sv = reinterpret_cast<const uint4 *>(Sa)[slot];
    const uint4 o0 = reinterpret_cast<const uint4 *>(So)[slot];
    const uint4 oyp = reinterpret_cast<const uint4 *>(So)[s_yp];
    const uint4 oym = reinterpret_cast<const uint4 *>(So)[s_ym];
    const uint4 ozp = reinterpret_cast<const uint4 *>(So)[s_zp];
    const uint4 ozm = reinterpret_cast<const uint4 *>(So)[s_zm];
    SlotK K;
    {
        const uint4 k0 = thr_t[0], k1 = thr_t[1], k2 = thr_t[2];
        K.lo[0] = k0.x; K.lo[1] = k0.y; K.lo[2] = k0.z; K.lo[3] = k0.w;
        K.lo[4] = k1.x; K.lo[5] = k1.y; K.lo[6] = k1.z; K.b3c = k1.w;
        K.nc = k2.x; K.ec = k2.y;
    }
    const uint32_t s[4] = {sv.x, sv.y, sv.z, sv.w};
    const uint32_t rr[4] = {r4.x, r4.y, r4.z, r4.w};
    const uint32_t v0[4] = {o0.x, o0.y, o0.z, o0.w};
    // second x-neighbour: m+1 for p = 1, m-1 for p = 0 (periodic within the row) — static renaming
    const uint32_t vB[4] = {P ? o0.y : o0.w, P ? o0.z : o0.x, P ? o0.w : o0.y, P ? o0.x : o0.z};
    const uint32_t vyp[4] = {oyp.x, oyp.y, oyp.z, oyp.w}, vym[4] = {oym.x, oym.y, oym.z, oym.w};
    const uint32_t vzp[4] = {ozp.x, ozp.y, ozp.z, ozp.w}, vzm[4] = {ozm.x, ozm.y, ozm.z, ozm.w};
    uint32_t out[4], w[4][3];
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const uint32_t u0 = xor3(s[e], v0[e], JA[e]), u1 = xor3(s[e], vB[e], JB[e]), u2 = xor3(s[e], vyp[e], Jyp[e]);
        const uint32_t u3 = xor3(s[e], vym[e], Jym[e]), u4 = xor3(s[e], vzp[e], Jzp[e]), u5 = xor3(s[e], vzm[e], Jzm[e]);
        if (!ENERGY) {
            out[e] = flip_word_k<BS>(s[e], amask, u0, u1, u2, u3, u4, u5, rr[e], K, one, mone);
        } else {
            uint32_t n0, n1, n2;
            const uint32_t acc = accept_word<BS>(u0, u1, u2, u3, u4, u5, ~(s[e] ^ amask), rr[e], K, one, mone, n0, n1, n2);
            out[e] = s[e] ^ acc;
            // post-flip unsatisfied count of this site: n if not flipped, 6 - n if flipped
            // 6 - n: bit0 = n0; bit1 = 1 for n in {0,3,4}; bit2 = 1 for n in {0,1,2}
            const uint32_t f1 = (~n2 & ~(n1 ^ n0)) | (n2 & ~n1 & ~n0);
            const uint32_t f2 = ~n2 & ~(n1 & n0);
            w[e][0] = n0;
            w[e][1] = (acc & f1) | (~acc & n1);
            w[e][2] = (acc & f2) | (~acc & n2);
        }
    }
    reinterpret_cast<uint4 *>(Sa)[slot] = make_uint4(out[0], out[1], out[2], out[3]);
    if (ENERGY) {
        uint32_t ab[4], cd[4], U[5];
        bs_sum<3>(w[0], w[1], ab);
        bs_sum<3>(w[2], w[3], cd);
        bs_sum<4>(ab, cd, U);
        // M: 8 words (4 new own-colour + 4 other-colour of the same row) -> 4 planes
        const uint32_t a1 = xor3(out[0], out[1], out[2]), c1 = maj3(out[0], out[1], out[2]);
        const uint32_t a2 = xor3(out[3], v0[0], v0[1]), c2 = maj3(out[3], v0[0], v0[1]);
        const uint32_t a3 = xor3(a1, a2, v0[2]), c3 = maj3(a1, a2, v0[2]);
        const uint32_t ones = a3 ^ v0[3], c4 = a3 & v0[3];
        const uint32_t t1 = xor3(c1, c2, c3), f1 = maj3(c1, c2, c3);
        const uint32_t twos = t1 ^ c4, f2 = t1 & c4;
        const uint32_t fours = f1 ^ f2, eights = f1 & f2;
        // red[plane][64 threads of the system]
#pragma unroll
        for (int k = 0; k < 5; ++k) red[k * 64] = U[k];
        red[5 * 64] = ones;
        red[6 * 64] = twos;
        red[7 * 64] = fours;
        red[8 * 64] = eights;
    }
}

// SPT = systems per thread (NT / G) when it is a compile-time constant (unrolled), 0 = run-time loop
// PT = false: the instantiation for launches without exchanges (all exchange code compiled out)
template <int SPT, bool BS, bool PT>
__global__ void __launch_bounds__(320, 2) k_ladder8_pmj(const __grid_constant__ Ladder8Args A)
{
    constexpr int N = 512, H = 256;
    extern __shared__ __align__(16) uint32_t smem[];
    const Dims &d = A.d;
    const int NT = d.NT;
    uint32_t *S = smem;                                    // [NT][2][64 slots][4]
    uint32_t *Jsm = S + NT * N;                            // [2][3][64 slots][4]
    uint4 *thr = reinterpret_cast<uint4 *>(Jsm + 3 * N);   // [NT][3] = SlotK: lo[7], b3c, nc, ec, 0, 0
    uint32_t *masks = reinterpret_cast<uint32_t *>(thr + NT * 3);     // [32]
    uint32_t *accs = masks + 32;                           // [MAX_NT] accepted swaps of this CTA per lower slot
    // exchange scratch (allocated only when pt_every > 0); later stages alias dead earlier ones
    uint32_t *red0 = accs + MAX_NT;                        // [NT][9][64]   stage-1 planes
    uint32_t *red1 = red0 + NT * PW1 * 64;                 // [NT][13][16]
    uint32_t *red2 = red0;                                 // [NT][17][4]   (red0 is dead after stage 2)
    uint32_t *red3 = red1;                                 // [NT][21][1]   (red1 is dead after stage 3)

    const int w = blockIdx.x / d.R, a = blockIdx.x % d.R;
    const int tid = threadIdx.x, nthr = blockDim.x;
    uint32_t *gS = A.spins + ((size_t)(w * d.R + a) * NT) * N;
    uint32_t *gOut = A.spins_out + ((size_t)(w * d.R + a) * NT) * N;
    const uint32_t *gJ = A.J + (size_t)w * 3 * N;

    // ---- load (global compact order -> slot order)
    for (int i = tid; i < NT * 128; i += nthr) {           // quads of all systems, both colours
        const int qq = i & 63, tc = i >> 6;                // tc = t*2 + colour
        reinterpret_cast<uint4 *>(S)[tc * 64 + slot_of_row(qq & 7, qq >> 3)] = reinterpret_cast<const uint4 *>(gS)[i];
    }
    for (int i = tid; i < 6 * 64; i += nthr) {             // [colour][d][quad]
        const int qq = i & 63, cd = i >> 6;
        reinterpret_cast<uint4 *>(Jsm)[cd * 64 + slot_of_row(qq & 7, qq >> 3)] = reinterpret_cast<const uint4 *>(gJ)[i];
    }
    for (int t = tid; t < NT; t += nthr) {                 // acceptance constants (see SlotK)
        uint32_t lo[7], hi[7], kw[10];
        for (int c = 0; c < 7; ++c) {
            const uint2 v = A.tab[t].c64[c];               // (0 - thr) as 64 bits
            lo[c] = v.x;
            hi[c] = v.y;
        }
        slotk_words<BS>(lo, hi, kw);
        thr[t * 3 + 0] = make_uint4(kw[0], kw[1], kw[2], kw[3]);
        thr[t * 3 + 1] = make_uint4(kw[4], kw[5], kw[6], kw[7]);
        thr[t * 3 + 2] = make_uint4(kw[8], kw[9], 0u, 0u);
    }
    if (tid < MAX_NT) accs[tid] = 0u;
    __syncthreads();

    // ---- thread geometry (colour independent)
    const int g = tid >> 6, pi = (tid >> 5) & 1, j = tid & 31;
    const int z = j >> 2, yy = j & 3, y = 2 * yy + ((pi + z) & 1);
    const int slot = pi * 32 + j, q = z * 8 + y;
    const int ob = (1 - pi) * 32;
    const int s_yp = ob + z * 4 + (((y + 1) & 7) >> 1), s_ym = ob + z * 4 + (((y + 7) & 7) >> 1);
    const int s_zp = ob + ((z + 1) & 7) * 4 + yy, s_zm = ob + ((z + 7) & 7) * 4 + yy;
    const bool active = g < A.G;
    const uint32_t amask = d.neg_h ? 0xffffffffu : 0u;
    const uint32_t wglob = (uint32_t)(w + (d.s_first >> 5));
    uint64_t exchange = A.exchange0;

    for (int sw = 0; sw < A.n_sweeps; ++sw) {
        const uint64_t sweep = A.sweep0 + (uint64_t)sw;
        const bool pt_due = PT && A.pt_every > 0 && ((sweep + 1) % (uint64_t)A.pt_every) == 0;
#pragma unroll 1
        for (int colour = 0; colour < 2; ++colour) {
            if (active) {
                const uint32_t time = 2u * (uint32_t)sweep + (uint32_t)colour;
                const int p = (colour + pi) & 1;
                const uint32_t *Jown = Jsm + (colour * 3) * H;
                const uint32_t *Joth = Jsm + ((1 - colour) * 3) * H;
                uint32_t JA[4], JB[4], Jyp[4], Jym[4], Jzp[4], Jzm[4];
                {
                    const uint4 jx = reinterpret_cast<const uint4 *>(Jown)[slot];
                    const uint4 jox = reinterpret_cast<const uint4 *>(Joth)[slot];
                    const uint4 jy = reinterpret_cast<const uint4 *>(Jown + H)[slot];
                    const uint4 joy = reinterpret_cast<const uint4 *>(Joth + H)[s_ym];
                    const uint4 jz = reinterpret_cast<const uint4 *>(Jown + 2 * H)[slot];
                    const uint4 joz = reinterpret_cast<const uint4 *>(Joth + 2 * H)[s_zm];
                    if (p) {       // neighbour at the same m is the -x one (its bond), at m+1 the +x one (own bond)
                        JA[0] = jox.x; JA[1] = jox.y; JA[2] = jox.z; JA[3] = jox.w;
                        JB[0] = jx.x; JB[1] = jx.y; JB[2] = jx.z; JB[3] = jx.w;
                    } else {       // neighbour at the same m is the +x one (own bond), at m-1 the -x one (its bond)
                        JA[0] = jx.x; JA[1] = jx.y; JA[2] = jx.z; JA[3] = jx.w;
                        JB[0] = jox.w; JB[1] = jox.x; JB[2] = jox.y; JB[3] = jox.z;
                    }
                    Jyp[0] = jy.x; Jyp[1] = jy.y; Jyp[2] = jy.z; Jyp[3] = jy.w;
                    Jym[0] = joy.x; Jym[1] = joy.y; Jym[2] = joy.z; Jym[3] = joy.w;
                    Jzp[0] = jz.x; Jzp[1] = jz.y; Jzp[2] = jz.z; Jzp[3] = jz.w;
                    Jzm[0] = joz.x; Jzm[1] = joz.y; Jzm[2] = joz.z; Jzm[3] = joz.w;
                }
                const bool want_energy = pt_due && colour == 1;
                auto body = [&](int t, const uint4 r_cur) {
                    uint32_t *Sa = S + t * N + colour * H;
                    const uint32_t *So = S + t * N + (1 - colour) * H;
                    uint32_t *red = red0 + (size_t)t * PW1 * 64 + (pi * 32 + j);
                    const uint4 *kt = thr + t * 3;
                    if (want_energy) {
                        if (p) half_sweep_quad<1, true, BS>(Sa, So, slot, s_yp, s_ym, s_zp, s_zm, JA, JB, Jyp, Jym, Jzp, Jzm,
                                                        r_cur, kt, amask, A.one, A.mone, red);
                        else   half_sweep_quad<0, true, BS>(Sa, So, slot, s_yp, s_ym, s_zp, s_zm, JA, JB, Jyp, Jym, Jzp, Jzm,
                                                        r_cur, kt, amask, A.one, A.mone, red);
                    } else {
                        if (p) half_sweep_quad<1, false, BS>(Sa, So, slot, s_yp, s_ym, s_zp, s_zm, JA, JB, Jyp, Jym, Jzp, Jzm,
                                                         r_cur, kt, amask, A.one, A.mone, red);
                        else   half_sweep_quad<0, false, BS>(Sa, So, slot, s_yp, s_ym, s_zp, s_zm, JA, JB, Jyp, Jym, Jzp, Jzm,
                                                         r_cur, kt, amask, A.one, A.mone, red);
                    }
                };
                if constexpr (SPT > 0) {
#pragma unroll 1
                    for (int i = 0; i < SPT; ++i) {
                        const int t = g + i * A.G;
                        body(t, philox_rk8((uint32_t)q, time, wglob, ctr3(3, a, t), A.rk));
                    }
                } else {
#pragma unroll 1
                    for (int t = g; t < NT; t += A.G)
                        body(t, philox_rk8((uint32_t)q, time, wglob, ctr3(3, a, t), A.rk));
                }
                // the two warps of this group share systems; other groups are independent
                asm volatile("bar.sync %0, 64;" ::"r"(g + 1) : "memory");
            }
        }
        if (pt_due) {
            __syncthreads();
            // ---- per-lane energies: three 4:1 bit-sliced adder stages, then one transpose per system
            reduce4<5, 4>(red0, red1, NT, 64, tid, nthr);
            __syncthreads();
            reduce4<7, 6>(red1, red2, NT, 16, tid, nthr);
            __syncthreads();
            reduce4<9, 8>(red2, red3, NT, 4, tid, nthr);
            __syncthreads();
            // ---- decisions and swaps: one WARP per pair.  The warp turns the count planes of its two systems into per-lane
            // integers itself (one bit transpose each), decides (lane l = sample 32 w + l) and, knowing the mask from its own
            // ballot, swaps the two configurations at once — no transpose phase, no barrier between decision and swap.
            const int e1 = (int)(exchange & 1u);
            const int npairs = (NT - e1) / 2;
            {
                const int lane = tid & 31, warp = tid >> 5, nwarp = nthr >> 5;
                for (int pair = warp; pair < npairs; pair += nwarp) {
                    const int t = e1 + 2 * pair;
                    const int s = w * 32 + lane;
                    const uint32_t v0 = transpose32(lane < 21 ? red3[t * 21 + lane] : 0u, lane);            // 11 planes of U, 10 of M
                    const uint32_t v1 = transpose32(lane < 21 ? red3[(t + 1) * 21 + lane] : 0u, lane);
                    const int U0 = (int)(v0 & 0x7ffu), U1 = (int)(v1 & 0x7ffu);
                    const int M0 = 2 * (int)((v0 >> 11) & 0x3ffu) - N, M1 = 2 * (int)((v1 >> 11) & 0x3ffu) - N;
                    const double Et = __dsub_rn((double)(2 * U0 - 3 * N), __dmul_rn(A.h, (double)M0));
                    const double Eu = __dsub_rn((double)(2 * U1 - 3 * N), __dmul_rn(A.h, (double)M1));
                    const double x = __dmul_rn(__dsub_rn(A.tab[t].beta, A.tab[t + 1].beta), __dsub_rn(Et, Eu));
                    const uint4 r = philox_rk8(0u, (uint32_t)exchange, (uint32_t)(s + d.s_first), ctr3(4, a, t), A.rk);
                    const bool accept = (x >= 0.0) || ((uint64_t)r.x < dexp64(A.exp_tab, -x));
                    const uint32_t mask = __ballot_sync(0xffffffffu, accept && s < d.n_samples);
                    if (lane == 0) { masks[pair] = mask; accs[t] += (uint32_t)__popc(mask); }
                    if (mask != 0u) {                                         // masked swap (layout independent: same slot in both systems)
#pragma unroll
                        for (int k = lane; k < 128; k += 32) {
                            uint4 *X = reinterpret_cast<uint4 *>(S + t * N) + k;
                            uint4 *Y = reinterpret_cast<uint4 *>(S + (t + 1) * N) + k;
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
            }
            if (sw == A.n_sweeps - 1) {
                // the launch ends here: publish the energies the decisions used, permuted like the configurations
                __syncthreads();                                              // masks of all pairs
                const int lane = tid & 31, warp = tid >> 5, nwarp = nthr >> 5;
                for (int t = warp; t < NT; t += nwarp) {
                    const int p = t - e1;
                    int src = t;
                    if (p >= 0 && (p >> 1) < npairs && ((masks[p >> 1] >> lane) & 1u)) src = (p & 1) ? t - 1 : t + 1;
                    // per-lane integers of both candidate systems (the transposes need the whole warp), then the lane's choice
                    const uint32_t vt = transpose32(lane < 21 ? red3[t * 21 + lane] : 0u, lane);
                    const int other = (p >= 0 && (p >> 1) < npairs) ? ((p & 1) ? t - 1 : t + 1) : t;
                    const uint32_t vo = transpose32(lane < 21 ? red3[other * 21 + lane] : 0u, lane);
                    const uint32_t v = src == t ? vt : vo;
                    const size_t o = ((size_t)(w * 32 + lane) * d.R + a) * NT + t;
                    A.U[o] = (int64_t)(v & 0x7ffu);
                    A.M[o] = 2 * (int)((v >> 11) & 0x3ffu) - N;
                }
            }
            exchange += 1;
            __syncthreads();
        }
    }
    __syncthreads();
    if (tid < NT && accs[tid]) atomicAdd(&A.pt_acc[tid], (unsigned long long)accs[tid]);

    // ---- write back (slot order -> global compact order)
    for (int i = tid; i < NT * 128; i += nthr) {
        const int qq = i & 63, tc = i >> 6;
        reinterpret_cast<uint4 *>(gOut)[i] = reinterpret_cast<const uint4 *>(S)[tc * 64 + slot_of_row(qq & 7, qq >> 3)];
    }
}

// ------------------------------------------------------------------------------- host side
static size_t ladder8_smem(int NT, bool with_pt)
{
    size_t b = (size_t)NT * 512 * 4 + 3 * 512 * 4 + (size_t)NT * 3 * sizeof(uint4) + 32 * 4 + MAX_NT * 4;
    if (with_pt) b += (size_t)NT * 4 * (PW1 * 64 + 13 * 16);
    return b;
}

bool ladder8_supported(const sg_ctx *c)
{
    const Dims &d = c->d;
    return c->path == SG_PATH_AUTO && c->kind == SG_PMJ && d.fast_accept && d.L == 8 &&
           ladder8_smem(d.NT, true) <= (size_t)113 * 1024;
}

// n_sweeps sweeps (global indices sweep0...) with the exchanges that fall due (pt_every; 0 = none).
// Returns kernels launched (1) or -1.  The caller advances its sweep / exchange counters.
int launch_ladder8_pmj(sg_ctx *c, uint64_t sweep0, uint64_t exchange0, int n_sweeps, int pt_every, uint32_t *spins_out)
{
    if (attr_needed(c, ATTR_LADDER8)) {
        bool ok = true;
        auto set = [&](auto kern) { ok = ok && cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 113 * 1024) == cudaSuccess; };
        set(k_ladder8_pmj<0, false, false>); set(k_ladder8_pmj<1, false, false>); set(k_ladder8_pmj<2, false, false>); set(k_ladder8_pmj<4, false, false>);
        set(k_ladder8_pmj<0, true, false>); set(k_ladder8_pmj<1, true, false>); set(k_ladder8_pmj<2, true, false>); set(k_ladder8_pmj<4, true, false>);
        set(k_ladder8_pmj<0, false, true>); set(k_ladder8_pmj<1, false, true>); set(k_ladder8_pmj<2, false, true>); set(k_ladder8_pmj<4, false, true>);
        set(k_ladder8_pmj<0, true, true>); set(k_ladder8_pmj<1, true, true>); set(k_ladder8_pmj<2, true, true>); set(k_ladder8_pmj<4, true, true>);
        if (!ok) return -1;
    }
    const Dims &d = c->d;
    Ladder8Args A;
    A.d = d;
    A.spins = c->spins;
    A.spins_out = spins_out ? spins_out : c->spins;
    A.J = c->J;
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
    int G = d.NT < 5 ? d.NT : 5;
    for (int gtry = G; gtry >= 1; --gtry)
        if (d.NT % gtry == 0) { G = gtry; break; }
    A.G = G;
    // whole-CTA phases assume complete warps; always launch 64*G threads (G <= 5 -> <= 320)
    const int threads = 64 * G;
    A.one = 1u;
    A.mone = 0xffffffffu;
    A.U = c->U;
    A.M = c->M;
    A.pt_acc = c->pt_acc;
    const size_t smem = ladder8_smem(d.NT, pt_every > 0);
    const int spt = d.NT % G == 0 ? d.NT / G : 0;
    const int grid = d.W * d.R;
    auto go = [&](auto kern) { kern<<<grid, threads, smem, c->stream>>>(A); };
    const bool pt = pt_every > 0;
#define SG_L8_PICK(SPTV)                                                                                        \
    do {                                                                                                        \
        if (d.bs_accept) { if (pt) go(k_ladder8_pmj<SPTV, true, true>); else go(k_ladder8_pmj<SPTV, true, false>); }   \
        else { if (pt) go(k_ladder8_pmj<SPTV, false, true>); else go(k_ladder8_pmj<SPTV, false, false>); }            \
    } while (0)
    if (spt == 4) SG_L8_PICK(4);
    else if (spt == 2) SG_L8_PICK(2);
    else if (spt == 1) SG_L8_PICK(1);
    else SG_L8_PICK(0);
#undef SG_L8_PICK
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace sg
