// sg_res32.cu — L = 32 (+-J) sweep kernel: ONE system (32768 word-sites = 128 KB) is resident in the
// shared memory of one SM for all sweeps of a launch (BASELINE.json config 5: 4 sweeps between exchanges),
// so the spin state crosses HBM once per launch (2 B per word-site and sweep at 4 sweeps) instead of
// once per half sweep; it arrives by eight 16 KB bulk-async copies (TMA) on one mbarrier.  The couplings of
// the packed word (shared by its R * NT = 128 systems, which are consecutive CTAs, so they stay in L2) stream
// through per-warp two-stage rings in shared memory, filled by bulk-async copies two warp steps ahead.
//
// Layout in shared memory = the canonical colour-compacted layout of global memory
// ([colour][z][y][16 words], one row = 64 B).  A warp owns 4 "diagonal pairs" of rows
// {(y, z), (y+1, z+1)} of one parity pi = (y+z)&1: the two rows of a quarter-warp are 33 rows apart,
// i.e. 16 banks, so every 128-bit shared access is conflict-free, and the row parity
// p = (colour + pi) & 1 that decides on which side the second x-neighbour sits is warp-uniform.
// Lane = 8*pair + 4*which + quad; the x-neighbour across a quad boundary comes from the adjacent lane.
//
// Exchange step (R12), split over two launches so that it costs no pass over the state: the launch that ends at an
// exchange point writes per-lane U, M (below); the NEXT launch decides the swap of its pair from those (one warp, 32
// lanes = 32 samples, the same decision in both CTAs of the pair) and, only for the lanes that swap, merges the
// partner's configuration into its own while loading ("swap on load").  State and energies are double-buffered
// (read spins_in / U_in, write spins_out / U) because the partner CTA needs this CTA's old configuration.
//
// Energy for the exchange step: in the last colour-1 half sweep every thread accumulates the
// post-flip unsatisfied-bond counts of its colour-1 sites (every bond has exactly one colour-1 end) and
// the spin words of both colours in bit-sliced registers; one warp transpose per plane turns them into
// per-lane integers U, M for the decision kernel.
#include "sg_accept.cuh"
#include "sg_device.cuh"
#include "sg_internal.h"

#include <type_traits>

namespace sg {

struct Res32Args {
    Dims d;
    const uint32_t *spins_in; // state before this launch (and before the pending exchange, if any)
    uint32_t *spins_out;      // state after it (a different buffer: a CTA may need its partner's OLD configuration)
    const uint4 *Jp;          // packed couplings (k_pack_J_res32)
    const int64_t *U_in;      // energies of the state in spins_in (read only if do_exchange)
    const int32_t *M_in;
    int64_t *U;               // energies of the state in spins_out (written only if want_energy)
    int32_t *M;
    const SlotTab *tab;       // beta per slot (exchange decision)
    const double *exp_tab;    // dexp64 table (R12)
    unsigned long long *pt_acc;
    double h;
    int do_exchange;          // apply exchange `exchange` (R12) to the loaded state before sweeping
    uint32_t exchange;
    uint32_t rk[20];
    uint64_t sweep0;          // global index of the first sweep of this launch
    int n_sweeps;
    int want_energy;          // write U, M of the final state
    uint32_t one, mone;
    uint32_t kc[MAX_NT][10];  // per slot: SlotK (lo[7], b3c, nc, ec); read through the constant bank with a uniform index
};

namespace {

constexpr int RL = 32, RN = RL * RL * RL, RH = RN / 2, RQ = RH / 4;   // 4096 quads per colour
constexpr int R_THREADS = 512, R_WARPS = R_THREADS / 32, R_ITERS = RQ / R_THREADS;   // 8 quads per thread and half sweep

// Couplings as the kernel consumes them ("packed" copy, built once per reset by k_pack_J_res32):
// Jp[w][colour][Z][warp&7][6][32 lanes] uint4 — for every warp step (colour, plane pair Z, row block)
// the six 4-word sets of each lane's quad, already in the order the update uses them
//   0: bond to the x-neighbour at the same compact m      1: bond to the other x-neighbour (m+1 / m-1)
//   2: +y (own)   3: -y (owned by row y-1)   4: +z (own)   5: -z (owned by row z-1)
// = one contiguous 3 KB chunk per warp step, fetched by ONE bulk-async copy (TMA) into the warp's own
// two-stage ring in shared memory; completion is tracked by an mbarrier per (warp, stage).
constexpr int CHUNK_U4 = 6 * 32, CHUNK_BYTES = CHUNK_U4 * 16;              // 3072 B
constexpr int CHUNKS_PER_WORD = 2 * 16 * 8;                                // colour, Z, row block
constexpr int N_STAGES = 2;

struct Quad6 {
    uint4 a, b, yp, ym, zp, zm;
};

// A thread's quad inside a z-plane pair is fixed for the whole launch (y, which row of the diagonal
// pair, quad within the row); only the plane pair Z = 0..15 changes from step to step.  All shared-memory
// addresses are 32-bit byte addresses: (thread constant) + 4096 * Z (warp-uniform).
struct Geo32 {
    uint32_t tb;                    // byte offset of the quad for Z = 0 inside one colour array (64 KB)
    uint32_t dyp, dym;              // byte deltas to the rows y+1, y-1 (periodic)
};

__device__ __forceinline__ Geo32 geo_of(int wj, int lane)
{
    const int pi = (wj >> 2) & 1, j = wj & 3;
    const int jj = lane >> 3, dd = (lane >> 2) & 1, m4 = lane & 3;
    const int y = (2 * (4 * j + jj) + pi + dd) & 31;
    Geo32 g;
    g.tb = (uint32_t)(128 * dd + 4 * y + m4) * 16u;
    g.dyp = (uint32_t)(64 * (((y + 1) & 31) - y));
    g.dym = (uint32_t)(64 * (((y + 31) & 31) - y));
    return g;
}

__device__ __forceinline__ uint4 lds128(uint32_t addr)
{
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
    return v;
}

__device__ __forceinline__ void sts128(uint32_t addr, const uint4 v)
{
    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}

__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "W_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra D_%=;\n\t"
        "bra W_%=;\n\t"
        "D_%=:\n\t}" ::"r"(bar), "r"(parity) : "memory");
}

// true in exactly one lane of a converged warp (elect.sync): the bulk-copy issue below stays a warp-uniform region —
// with `lane == 0` ptxas wraps the uniform-operand UBLKCP in an ELECT loop over the active lanes
__device__ __forceinline__ bool elect_one()
{
    uint32_t pred;
    asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
    return pred != 0;
}

// one lane: arm the barrier with the byte count and start the bulk copy global -> shared
__device__ __forceinline__ void bulk_load(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}

// sa / so: byte addresses of the own-colour / other-colour array; qb: byte offset of the quad in them
template <int P, bool ENERGY, bool BS>
__device__ __forceinline__ void quad_update(uint32_t sa, uint32_t so, uint32_t qb, const Geo32 &g, const Quad6 &Jq,
                                            const uint4 r4, const SlotK &K, uint32_t amask, uint32_t one, uint32_t mone,
                                            int lane, uint32_t (&accU)[8], uint32_t (&accM)[7], uint4 *gst)
{
    const uint4 sv = lds128(sa + qb);
    const uint4 o0 = lds128(so + qb);
    const uint4 oyp = lds128(so + qb + g.dyp), oym = lds128(so + qb + g.dym);
    const uint4 ozp = lds128(so + ((qb + 2048u) & 0xffffu)), ozm = lds128(so + ((qb - 2048u) & 0xffffu));
    // word of the adjacent quad of the same row (periodic): m+1 for p = 1, m-1 for p = 0
    const int src = (lane & ~3) | ((lane + (P ? 1 : 3)) & 3);
    const uint32_t side = __shfl_sync(0xffffffffu, P ? o0.x : o0.w, src);
    const uint32_t s[4] = {sv.x, sv.y, sv.z, sv.w};
    const uint32_t rr[4] = {r4.x, r4.y, r4.z, r4.w};
    const uint32_t v0[4] = {o0.x, o0.y, o0.z, o0.w};
    // second x-neighbour: at m+1 for p = 1, at m-1 for p = 0 (the packed couplings are already in this order)
    uint32_t vB[4];
    if (P) { vB[0] = o0.y; vB[1] = o0.z; vB[2] = o0.w; vB[3] = side; }
    else   { vB[0] = side; vB[1] = o0.x; vB[2] = o0.y; vB[3] = o0.z; }
    const uint32_t JA[4] = {Jq.a.x, Jq.a.y, Jq.a.z, Jq.a.w}, JB[4] = {Jq.b.x, Jq.b.y, Jq.b.z, Jq.b.w};
    const uint32_t Jyp[4] = {Jq.yp.x, Jq.yp.y, Jq.yp.z, Jq.yp.w}, Jym[4] = {Jq.ym.x, Jq.ym.y, Jq.ym.z, Jq.ym.w};
    const uint32_t Jzp[4] = {Jq.zp.x, Jq.zp.y, Jq.zp.z, Jq.zp.w}, Jzm[4] = {Jq.zm.x, Jq.zm.y, Jq.zm.z, Jq.zm.w};
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
            // post-flip unsatisfied count: n if not flipped, 6 - n if flipped
            // 6 - n: bit0 = n0; bit1 = 1 for n in {0,3,4}; bit2 = 1 for n in {0,1,2}
            const uint32_t f1 = (~n2 & ~(n1 ^ n0)) | (n2 & ~n1 & ~n0);
            const uint32_t f2 = ~n2 & ~(n1 & n0);
            w[e][0] = n0;
            w[e][1] = (acc & f1) | (~acc & n1);
            w[e][2] = (acc & f2) | (~acc & n2);
        }
    }
    sts128(sa + qb, make_uint4(out[0], out[1], out[2], out[3]));
    if (gst) {
        // last half sweep of the launch (colour 1): this quad and the colour-0 quad at the same index are final, so they
        // go to global memory from the registers now and the write-back overlaps the rest of the half sweep
        gst[RQ] = make_uint4(out[0], out[1], out[2], out[3]);
        gst[0] = o0;
    }
    if (ENERGY) {
        uint32_t ab[4], cd[4], U5[5];
        bs_sum<3>(w[0], w[1], ab);
        bs_sum<3>(w[2], w[3], cd);
        bs_sum<4>(ab, cd, U5);
        bs_add(accU, U5);
        // M: 4 new own-colour words + the 4 other-colour words of the same quad index -> 4 planes
        const uint32_t a1 = xor3(out[0], out[1], out[2]), c1 = maj3(out[0], out[1], out[2]);
        const uint32_t a2 = xor3(out[3], v0[0], v0[1]), c2 = maj3(out[3], v0[0], v0[1]);
        const uint32_t a3 = xor3(a1, a2, v0[2]), c3 = maj3(a1, a2, v0[2]);
        const uint32_t ones = a3 ^ v0[3], c4 = a3 & v0[3];
        const uint32_t t1 = xor3(c1, c2, c3), f1 = maj3(c1, c2, c3);
        const uint32_t twos = t1 ^ c4, f2 = t1 & c4;
        const uint32_t M4[4] = {ones, twos, f1 ^ f2, f1 & f2};
        bs_add(accM, M4);
    }
}

template <bool BS>
__global__ void __launch_bounds__(R_THREADS, 1) k_res32_pmj(const __grid_constant__ Res32Args A)
{
    extern __shared__ __align__(128) uint32_t smem[];
    uint4 *S4 = reinterpret_cast<uint4 *>(smem);                           // [2][RQ]                  128 KB
    uint4 *ring = S4 + 2 * RQ;                                             // [16 warps][2 stages][6][32] 96 KB
    uint64_t *bars = reinterpret_cast<uint64_t *>(ring + R_WARPS * N_STAGES * CHUNK_U4);   // [16][2]
    uint64_t *sysbar_p = bars + R_WARPS * N_STAGES;                        // [8] load barriers of the system: one per 16 KB chunk
    int *sUM = reinterpret_cast<int *>(sysbar_p + 8);                      // [2][32], then [64]: swap mask of this CTA
    const Dims &d = A.d;
    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);        // warp-uniform for the compiler: uniform datapath
    const int t = blockIdx.x, a = blockIdx.y, w = blockIdx.z;      // x fastest: the 128 systems of a word are consecutive CTAs
    const int sys = (w * d.R + a) * d.NT + t;
    const uint4 *gS = reinterpret_cast<const uint4 *>(A.spins_in + (size_t)sys * RN);
    uint4 *gO = reinterpret_cast<uint4 *>(A.spins_out + (size_t)sys * RN);
    const int zhalf = warp >> 3, wj = warp & 7;
    // chunk of (colour, Z) for this warp: Jp_w + ((colour * 16 + Z) * 8 + wj) * CHUNK_U4
    const uint4 *Jpw = A.Jp + ((size_t)w * CHUNKS_PER_WORD + wj) * CHUNK_U4;
    const uint32_t S_s = smem_u32(S4);
    const uint32_t ring_s = smem_u32(ring + warp * N_STAGES * CHUNK_U4), bar_s = smem_u32(bars + warp * N_STAGES);

    const int n_half = 2 * A.n_sweeps;
    // step (hs, it) of this warp: half sweep hs, iteration it = 0..7, plane pair Z = 2 it + zhalf, stage it & 1
    auto issue = [&](int hs, int it) {          // lane 0 only
        const int colour = hs & 1, Z = 2 * it + zhalf, st = it & 1;
        bulk_load(ring_s + st * CHUNK_BYTES, Jpw + (size_t)((colour * 16 + Z) * 8) * CHUNK_U4, CHUNK_BYTES, bar_s + st * 8);
    };
    if (lane == 0) {
        mbar_init(bar_s, 1);
        mbar_init(bar_s + 8, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        issue(0, 0);
        issue(0, 1);
    }

    // ---- load the system (contiguous 128 KB): eight 16 KB bulk-async copies, each on its own mbarrier, issued in the
    // order the first half sweep needs them (chunk k = colour k >> 2, planes 8 (k & 3) .. 8 (k & 3) + 7): the first
    // warp steps start as soon as their three chunks have landed instead of after the whole system
    const uint32_t sysbar = smem_u32(sysbar_p);
    if (tid == 0) {
#pragma unroll
        for (int i = 0; i < 8; ++i) mbar_init(sysbar + 8 * i, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        constexpr int order[8] = {0, 4, 7, 5, 1, 6, 2, 3};
#pragma unroll
        for (int i = 0; i < 8; ++i)
            bulk_load(S_s + order[i] * 16384, reinterpret_cast<const char *>(gS) + order[i] * 16384, 16384, sysbar + 8 * order[i]);
    }
    if (tid < 64) sUM[tid] = 0;
    // ---- pending exchange: decide the swap of this slot's pair (warp 0; lane l = sample 32 w + l)
    int partner = -1;
    if (A.do_exchange) {
        const int e1 = (int)(A.exchange & 1u), p = t - e1;
        if (p >= 0 && (p >> 1) < (d.NT - e1) / 2) partner = (p & 1) ? t - 1 : t + 1;
    }
    if (warp == 0) {
        uint32_t mask = 0u;
        if (partner >= 0) {
            const int tl = partner < t ? partner : t;               // lower slot of the pair
            const int smp = w * 32 + lane;
            const size_t o = ((size_t)smp * d.R + a) * d.NT + tl;
            const double Et = __dsub_rn((double)(2 * A.U_in[o] - 3 * (int64_t)RN), __dmul_rn(A.h, (double)A.M_in[o]));
            const double Eu = __dsub_rn((double)(2 * A.U_in[o + 1] - 3 * (int64_t)RN), __dmul_rn(A.h, (double)A.M_in[o + 1]));
            const double x = __dmul_rn(__dsub_rn(A.tab[tl].beta, A.tab[tl + 1].beta), __dsub_rn(Et, Eu));
            const uint4 r = philox_rk8(0u, A.exchange, (uint32_t)(smp + d.s_first), ctr3(4, a, tl), A.rk);
            const bool accept = (x >= 0.0) || ((uint64_t)r.x < dexp64(A.exp_tab, -x));
            mask = __ballot_sync(0xffffffffu, accept && smp < d.n_samples);
            if (lane == 0 && tl == t && mask) atomicAdd(&A.pt_acc[tl], (unsigned long long)__popc(mask));
        }
        if (lane == 0) sUM[64] = (int)mask;
    }

    SlotK K;                                                // block-uniform: stays in uniform registers / the constant bank
#pragma unroll
    for (int c = 0; c < 7; ++c) K.lo[c] = A.kc[t][c];
    K.b3c = A.kc[t][7];
    K.nc = A.kc[t][8];
    K.ec = A.kc[t][9];
    const uint32_t amask = d.neg_h ? 0xffffffffu : 0u;
    const uint32_t wglob = (uint32_t)(w + (d.s_first >> 5));
    const uint32_t c3 = ctr3(3, a, t);
    const Geo32 geo = geo_of(wj, lane);
    const int pi = (wj >> 2) & 1;
    __syncthreads();                                        // barriers initialised, sUM zeroed, swap mask known
    {
        const uint32_t xmask = (uint32_t)sUM[64];           // block-uniform
        if (xmask) {                                        // swap on load: take the partner's bits in the swapping lanes
#pragma unroll
            for (int i = 0; i < 8; ++i) mbar_wait(sysbar + 8 * i, 0u);     // the whole system has landed
            const uint4 *gP = reinterpret_cast<const uint4 *>(A.spins_in + (size_t)(sys - t + partner) * RN);
            constexpr int LUT_SEL = (0xF0 & 0x55) | (0xCC & 0xAA);           // c ? b : a
#pragma unroll 4
            for (int i = tid; i < 2 * RQ; i += R_THREADS) {
                const uint4 v = S4[i], pv = gP[i];
                S4[i] = make_uint4(lop3<LUT_SEL>(v.x, pv.x, xmask), lop3<LUT_SEL>(v.y, pv.y, xmask),
                                   lop3<LUT_SEL>(v.z, pv.z, xmask), lop3<LUT_SEL>(v.w, pv.w, xmask));
            }
            __syncthreads();
        }
    }

    auto half_sweep = [&](auto P_tag, auto E_tag, int hs) {
        constexpr int P = decltype(P_tag)::value;
        constexpr bool ENERGY = decltype(E_tag)::value;
        const int colour = hs & 1;
        const uint32_t time = 2u * (uint32_t)(A.sweep0 + (uint64_t)(hs >> 1)) + (uint32_t)colour;
        const uint32_t sa = S_s + (uint32_t)colour * 65536u, so = S_s + (uint32_t)(1 - colour) * 65536u;
        uint32_t accU[8], accM[7];                          // live in the ENERGY instantiations only
#pragma unroll
        for (int k = 0; k < 8; ++k) accU[k] = 0;
#pragma unroll
        for (int k = 0; k < 7; ++k) accM[k] = 0;
#pragma unroll 4
        for (int it = 0; it < R_ITERS; ++it) {
            const int st = it & 1;
            if (hs == 0) {                                  // first half sweep (colour 0): the chunks this step touches have landed?
                const int Z = 2 * it + zhalf;
                mbar_wait(sysbar + 8u * (uint32_t)(Z >> 2), 0u);                             // colour 0, planes 2 Z, 2 Z + 1
                mbar_wait(sysbar + 8u * (uint32_t)(4 + (((2 * Z + 31) & 31) >> 3)), 0u);     // colour 1, plane 2 Z - 1
                mbar_wait(sysbar + 8u * (uint32_t)(4 + (((2 * Z + 2) & 31) >> 3)), 0u);      // colour 1, plane 2 Z + 2
            }
            mbar_wait(bar_s + st * 8, (uint32_t)(it >> 1) & 1u);      // use (8 hs + it) / 2 of the stage: parity = bit 1 of it
            const uint32_t jc = ring_s + st * CHUNK_BYTES + lane * 16;
            Quad6 Jq;
            Jq.a = lds128(jc);
            Jq.b = lds128(jc + 512);
            Jq.yp = lds128(jc + 1024);
            Jq.ym = lds128(jc + 1536);
            Jq.zp = lds128(jc + 2048);
            Jq.zm = lds128(jc + 2560);
            const uint32_t qb = geo.tb + 4096u * (uint32_t)(2 * it + zhalf);
            quad_update<P, ENERGY, BS>(sa, so, qb, geo, Jq, philox_rk8(qb >> 4, time, wglob, c3, A.rk), K, amask, A.one,
                                   A.mone, lane, accU, accM, hs == n_half - 1 ? gO + (qb >> 4) : nullptr);
            // Refill the stage two steps ahead only now: every lane has CONSUMED its coupling registers, so the
            // shared-memory loads of the stage have completed (a load that is merely issued could still be in the
            // LSU queue when the bulk copy, which runs on a different engine, overwrites the stage).
            __syncwarp();
            if (elect_one()) {
                if (it + 2 < R_ITERS) issue(hs, it + 2);
                else if (hs + 1 < n_half) issue(hs + 1, it + 2 - R_ITERS);
            }
        }
        if constexpr (ENERGY) {                             // per-lane totals of this warp -> CTA totals
            const uint32_t totU = bs_warp_total(accU, 8, lane);
            const uint32_t totM = bs_warp_total(accM, 7, lane);
            atomicAdd(&sUM[lane], (int)totU);
            atomicAdd(&sUM[32 + lane], (int)totM);
        }
    };
    using T0 = std::integral_constant<int, 0>;
    using T1 = std::integral_constant<int, 1>;
#pragma unroll 1
    for (int hs = 0; hs < n_half; ++hs) {
        const int p = ((hs & 1) + pi) & 1;                  // warp-uniform row parity of this half sweep
        if (A.want_energy && hs == n_half - 1) {
            if (p) half_sweep(T1{}, std::true_type{}, hs);
            else   half_sweep(T0{}, std::true_type{}, hs);
        } else {
            if (p) half_sweep(T1{}, std::false_type{}, hs);
            else   half_sweep(T0{}, std::false_type{}, hs);
        }
        __syncthreads();
    }

    if (A.want_energy) {                                    // (the loop ended with a __syncthreads)
        if (tid < 32) {
            const size_t o = ((size_t)(w * 32 + tid) * d.R + a) * d.NT + t;
            A.U[o] = (int64_t)sUM[tid];
            A.M[o] = 2 * sUM[32 + tid] - RN;
        }
    }

    // (the state went back to global memory quad by quad during the last half sweep, see quad_update; a bulk-async
    // store at this point would hold the CTA until its completion — measured slower, as was a plain store loop)
}

// canonical couplings J[w][colour][dir][H] -> packed copy (see above); one thread per packed uint4
__global__ void __launch_bounds__(256) k_pack_J_res32(Dims d, const uint32_t *__restrict__ J, uint4 *__restrict__ Jp)
{
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long long)d.W * CHUNKS_PER_WORD * CHUNK_U4) return;
    const int lane = (int)(idx & 31), arr = (int)((idx >> 5) % 6);
    long long ch = idx / CHUNK_U4;
    const int wj = (int)(ch & 7);   ch >>= 3;
    const int Z = (int)(ch & 15);   ch >>= 4;
    const int colour = (int)(ch & 1);
    const int w = (int)(ch >> 1);
    const int pi = (wj >> 2) & 1, j = wj & 3;
    const int jj = lane >> 3, dd = (lane >> 2) & 1, m4 = lane & 3;
    const int y = (2 * (4 * j + jj) + pi + dd) & 31, z = 2 * Z + dd;
    const int p = (colour + pi) & 1;
    const uint32_t *Jown = J + ((size_t)(w * 2 + colour) * 3) * RH;
    const uint32_t *Joth = J + ((size_t)(w * 2 + 1 - colour) * 3) * RH;
    const int row = z * 32 + y;
    uint32_t v[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const int m = 4 * m4 + e;
        switch (arr) {
        case 0: v[e] = p ? Joth[row * 16 + m] : Jown[row * 16 + m]; break;                   // same m: -x bond (p=1) / +x own bond (p=0)
        case 1: v[e] = p ? Jown[row * 16 + m] : Joth[row * 16 + ((m + 15) & 15)]; break;     // m+1: own +x bond / m-1: its +x bond
        case 2: v[e] = Jown[RH + row * 16 + m]; break;
        case 3: v[e] = Joth[RH + (z * 32 + ((y + 31) & 31)) * 16 + m]; break;
        case 4: v[e] = Jown[2 * RH + row * 16 + m]; break;
        default: v[e] = Joth[2 * RH + (((z + 31) & 31) * 32 + y) * 16 + m]; break;
        }
    }
    Jp[idx] = make_uint4(v[0], v[1], v[2], v[3]);
}

constexpr size_t RES32_SMEM = (size_t)RN * 4 + (size_t)R_WARPS * N_STAGES * CHUNK_BYTES + R_WARPS * N_STAGES * 8 + 8 * 8 + 68 * 4;

}  // namespace

size_t res32_packed_bytes(int W) { return (size_t)W * CHUNKS_PER_WORD * CHUNK_BYTES; }

bool res32_supported(const sg_ctx *c)
{
    const Dims &d = c->d;
    return c->path == SG_PATH_AUTO && c->kind == SG_PMJ && d.fast_accept && d.L == 32 && c->Jp != nullptr;
}

// packed copy of the couplings (after every k_init_J_pmj)
int launch_pack_J_res32(sg_ctx *c)
{
    const Dims &d = c->d;
    const long long n = (long long)d.W * CHUNKS_PER_WORD * CHUNK_U4;
    k_pack_J_res32<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(d, c->J, c->Jp);
    return 1;
}

// n_sweeps consecutive sweeps from global sweep index sweep0; want_energy: also write U, M of the final
// state (fresh energies for the exchange step).  Returns kernels launched (1) or -1.
int launch_res32_pmj(sg_ctx *c, uint64_t sweep0, int n_sweeps, bool want_energy, bool do_exchange, uint64_t exchange)
{
    if (attr_needed(c, ATTR_RES32)) {
        if (cudaFuncSetAttribute(k_res32_pmj<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RES32_SMEM) != cudaSuccess ||
            cudaFuncSetAttribute(k_res32_pmj<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RES32_SMEM) != cudaSuccess)
            return -1;
    }
    const Dims &d = c->d;
    Res32Args A;
    A.d = d;
    A.spins_in = c->spins;
    A.spins_out = c->spins_alt;
    A.Jp = c->Jp;
    A.U_in = c->U;
    A.M_in = c->M;
    A.U = c->U_alt;
    A.M = c->M_alt;
    A.tab = c->tab;
    A.exp_tab = c->exp64_tab;
    A.pt_acc = c->pt_acc;
    A.h = c->h;
    A.do_exchange = do_exchange ? 1 : 0;
    A.exchange = (uint32_t)exchange;
    for (int r = 0; r < 10; ++r) {
        A.rk[2 * r] = d.k0 + (uint32_t)r * 0x9E3779B9u;
        A.rk[2 * r + 1] = d.k1 + (uint32_t)r * 0xBB67AE85u;
    }
    A.sweep0 = sweep0;
    A.n_sweeps = n_sweeps;
    A.want_energy = want_energy ? 1 : 0;
    A.one = 1u;
    A.mone = 0xffffffffu;
    for (int t = 0; t < d.NT; ++t) {                        // SlotK of sg_accept.cuh from the host threshold table
        uint32_t lo[7], hi[7];
        for (int code = 0; code < 7; ++code) {
            const uint64_t neg = (uint64_t)0 - c->thr[((size_t)t * 7 + (code >> 1)) * 2 + (1 - (code & 1))];
            lo[code] = (uint32_t)neg;
            hi[code] = (uint32_t)(neg >> 32);
        }
        if (d.bs_accept) slotk_words<true>(lo, hi, A.kc[t]);
        else slotk_words<false>(lo, hi, A.kc[t]);
    }
    if (d.bs_accept) k_res32_pmj<true><<<dim3(d.NT, d.R, d.W), R_THREADS, RES32_SMEM, c->stream>>>(A);
    else k_res32_pmj<false><<<dim3(d.NT, d.R, d.W), R_THREADS, RES32_SMEM, c->stream>>>(A);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace sg
