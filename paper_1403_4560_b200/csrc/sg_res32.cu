// sg_res32.cu — L = 32 (+-J) sweep kernel: ONE system (32768 word-sites = 128 KB) is resident in the
// shared memory of one SM for all sweeps of a launch (BASELINE.json config 5: 4 sweeps between exchanges),
// so the spin state crosses HBM once per launch (2 B per word-site and sweep at 4 sweeps) instead of
// once per half sweep.  The couplings of the packed word (384 KB, shared by its R * NT = 128 systems,
// which are consecutive CTAs) are streamed from L2 through registers, one quad ahead.
//
// Layout in shared memory = the canonical colour-compacted layout of global memory
// ([colour][z][y][16 words], one row = 64 B).  A warp owns 4 "diagonal pairs" of rows
// {(y, z), (y+1, z+1)} of one parity pi = (y+z)&1: the two rows of a quarter-warp are 33 rows apart,
// i.e. 16 banks, so every 128-bit shared access is conflict-free, and the row parity
// p = (colour + pi) & 1 that decides on which side the second x-neighbour sits is warp-uniform.
// Lane = 8*pair + 4*which + quad; the x-neighbour across a quad boundary comes from the adjacent lane.
//
// Energy for the exchange step (R12): in the last colour-1 half sweep every thread accumulates the
// post-flip unsatisfied-bond counts of its colour-1 sites (every bond has exactly one colour-1 end) and
// the spin words of both colours in bit-sliced registers; one warp transpose per plane turns them into
// per-lane integers U, M for the decision kernel.
#include "sg_accept.cuh"
#include "sg_device.cuh"
#include "sg_internal.h"

namespace sg {

struct Res32Args {
    Dims d;
    uint32_t *spins;
    const uint32_t *J;
    const SlotTab *tab;
    int64_t *U;
    int32_t *M;
    uint32_t rk[20];
    uint64_t sweep0;          // global index of the first sweep of this launch
    int n_sweeps;
    int want_energy;          // write U, M of the final state
    uint32_t one, mone;
};

namespace {

constexpr int RL = 32, RN = RL * RL * RL, RH = RN / 2, RQ = RH / 4;   // 4096 quads per colour
constexpr int R_THREADS = 512, R_WARPS = R_THREADS / 32, R_ITERS = RQ / R_THREADS;   // 8 quads per thread and half sweep

struct Quad6 {
    uint4 x, y, z, ox, oy, oz;     // own +x +y +z bonds; other colour's +x (same row), +y (row y-1), +z (row z-1)
};

struct Geo32 {
    int q, q_yp, q_ym, q_zp, q_zm;  // uint4 indices inside one colour array
    int p;
};

// task (0..127) of a warp and lane -> quad and its neighbour rows
__device__ __forceinline__ Geo32 geo_of(int task, int lane, int colour)
{
    const int Z = task >> 3, pi = (task >> 2) & 1, j = task & 3;
    const int jj = lane >> 3, dd = (lane >> 2) & 1, m4 = lane & 3;
    const int y = (2 * (4 * j + jj) + pi + dd) & 31, z = 2 * Z + dd;
    Geo32 g;
    g.p = (colour + pi) & 1;
    g.q = (z * 32 + y) * 4 + m4;
    g.q_yp = (z * 32 + ((y + 1) & 31)) * 4 + m4;
    g.q_ym = (z * 32 + ((y + 31) & 31)) * 4 + m4;
    g.q_zp = (((z + 1) & 31) * 32 + y) * 4 + m4;
    g.q_zm = (((z + 31) & 31) * 32 + y) * 4 + m4;
    return g;
}

__device__ __forceinline__ Quad6 load_J(const uint4 *__restrict__ Jw, int colour, const Geo32 &g)
{
    const uint4 *Jown = Jw + (size_t)colour * 3 * RQ;
    const uint4 *Joth = Jw + (size_t)(1 - colour) * 3 * RQ;
    Quad6 r;
    r.x = __ldg(Jown + g.q);
    r.y = __ldg(Jown + RQ + g.q);
    r.z = __ldg(Jown + 2 * RQ + g.q);
    r.ox = __ldg(Joth + g.q);
    r.oy = __ldg(Joth + RQ + g.q_ym);
    r.oz = __ldg(Joth + 2 * RQ + g.q_zm);
    return r;
}

template <int P, bool ENERGY>
__device__ __forceinline__ void quad_update(uint4 *__restrict__ Sa, const uint4 *__restrict__ So, const Geo32 &g,
                                            const Quad6 &Jq, const uint4 r4, const SlotK &K, uint32_t amask,
                                            uint32_t one, uint32_t mone, int lane, uint32_t (&accU)[8],
                                            uint32_t (&accM)[7])
{
    const uint4 sv = Sa[g.q];
    const uint4 o0 = So[g.q];
    const uint4 oyp = So[g.q_yp], oym = So[g.q_ym], ozp = So[g.q_zp], ozm = So[g.q_zm];
    // word of the adjacent quad of the same row (periodic): m+1 for p = 1, m-1 for p = 0
    const int src = (lane & ~3) | ((lane + (P ? 1 : 3)) & 3);
    const uint32_t side = __shfl_sync(0xffffffffu, P ? o0.x : o0.w, src);
    const uint32_t s[4] = {sv.x, sv.y, sv.z, sv.w};
    const uint32_t rr[4] = {r4.x, r4.y, r4.z, r4.w};
    const uint32_t v0[4] = {o0.x, o0.y, o0.z, o0.w};
    uint32_t vB[4], JA[4], JB[4];
    if (P) {       // same m: the -x neighbour (its bond); m+1: the +x neighbour (own bond)
        vB[0] = o0.y; vB[1] = o0.z; vB[2] = o0.w; vB[3] = side;
        JA[0] = Jq.ox.x; JA[1] = Jq.ox.y; JA[2] = Jq.ox.z; JA[3] = Jq.ox.w;
        JB[0] = Jq.x.x; JB[1] = Jq.x.y; JB[2] = Jq.x.z; JB[3] = Jq.x.w;
    } else {       // same m: the +x neighbour (own bond); m-1: the -x neighbour (its bond)
        const uint32_t jside = __shfl_sync(0xffffffffu, Jq.ox.w, src);
        vB[0] = side; vB[1] = o0.x; vB[2] = o0.y; vB[3] = o0.z;
        JA[0] = Jq.x.x; JA[1] = Jq.x.y; JA[2] = Jq.x.z; JA[3] = Jq.x.w;
        JB[0] = jside; JB[1] = Jq.ox.x; JB[2] = Jq.ox.y; JB[3] = Jq.ox.z;
    }
    const uint32_t Jyp[4] = {Jq.y.x, Jq.y.y, Jq.y.z, Jq.y.w}, Jym[4] = {Jq.oy.x, Jq.oy.y, Jq.oy.z, Jq.oy.w};
    const uint32_t Jzp[4] = {Jq.z.x, Jq.z.y, Jq.z.z, Jq.z.w}, Jzm[4] = {Jq.oz.x, Jq.oz.y, Jq.oz.z, Jq.oz.w};
    const uint32_t vyp[4] = {oyp.x, oyp.y, oyp.z, oyp.w}, vym[4] = {oym.x, oym.y, oym.z, oym.w};
    const uint32_t vzp[4] = {ozp.x, ozp.y, ozp.z, ozp.w}, vzm[4] = {ozm.x, ozm.y, ozm.z, ozm.w};
    uint32_t out[4], w[4][3];
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        uint32_t n0, n1, n2;
        const uint32_t acc = accept_word(xor3(s[e], v0[e], JA[e]), xor3(s[e], vB[e], JB[e]), xor3(s[e], vyp[e], Jyp[e]),
                                         xor3(s[e], vym[e], Jym[e]), xor3(s[e], vzp[e], Jzp[e]),
                                         xor3(s[e], vzm[e], Jzm[e]), ~(s[e] ^ amask), rr[e], K, one, mone, n0, n1, n2);
        out[e] = s[e] ^ acc;
        if (ENERGY) {
            // post-flip unsatisfied count: n if not flipped, 6 - n if flipped
            // 6 - n: bit0 = n0; bit1 = 1 for n in {0,3,4}; bit2 = 1 for n in {0,1,2}
            const uint32_t f1 = (~n2 & ~(n1 ^ n0)) | (n2 & ~n1 & ~n0);
            const uint32_t f2 = ~n2 & ~(n1 & n0);
            w[e][0] = n0;
            w[e][1] = (acc & f1) | (~acc & n1);
            w[e][2] = (acc & f2) | (~acc & n2);
        }
    }
    Sa[g.q] = make_uint4(out[0], out[1], out[2], out[3]);
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

__global__ void __launch_bounds__(R_THREADS, 1) k_res32_pmj(const __grid_constant__ Res32Args A)
{
    extern __shared__ __align__(16) uint32_t smem[];
    uint4 *S4 = reinterpret_cast<uint4 *>(smem);               // [2][RQ]
    int *sUM = reinterpret_cast<int *>(smem + RN);              // [2][32]
    const Dims &d = A.d;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int sys = blockIdx.x;
    const int t = sys % d.NT, a = (sys / d.NT) % d.R, w = sys / (d.NT * d.R);
    uint4 *gS = reinterpret_cast<uint4 *>(A.spins + (size_t)sys * RN);
    const uint4 *Jw = reinterpret_cast<const uint4 *>(A.J + (size_t)w * 3 * RN);

    // ---- load the system (contiguous 128 KB)
#pragma unroll 8
    for (int i = 0; i < 2 * RQ / R_THREADS; ++i) S4[i * R_THREADS + tid] = gS[i * R_THREADS + tid];
    if (tid < 64) sUM[tid] = 0;

    SlotK K;
    {
        uint32_t zc[7];
#pragma unroll
        for (int c = 0; c < 7; ++c) {
            const uint2 v = A.tab[t].c64[c];               // (0 - thr) as 64 bits: hi = 0 only for thr = 0
            K.lo[c] = v.x;
            zc[c] = v.y == 0u ? 1u : 0u;
        }
        K.b3c = zc[3] - 1u;
        K.nc = zc[1] + zc[5] - 1u;
        K.ec = zc[0] + zc[2] + zc[4] + zc[6] - 2u;
    }
    const uint32_t amask = d.neg_h ? 0xffffffffu : 0u;
    const uint32_t wglob = (uint32_t)(w + (d.s_first >> 5));
    const uint32_t c3 = ctr3(3, a, t);
    uint32_t accU[8], accM[7];
#pragma unroll
    for (int k = 0; k < 8; ++k) accU[k] = 0;
#pragma unroll
    for (int k = 0; k < 7; ++k) accM[k] = 0;
    __syncthreads();

    // ---- flat loop over (sweep, colour, iteration); couplings of the next step are loaded one step ahead.
    // Colour 1 walks the tasks in reverse so that the most recently read coupling lines are still in L1.
    const int n_steps = A.n_sweeps * 2 * R_ITERS;
    auto task_of = [&](int step) {
        const int colour = (step / R_ITERS) & 1, it = step % R_ITERS;
        const int task = it * R_WARPS + warp;
        return colour ? 127 - task : task;
    };
    Geo32 g = geo_of(task_of(0), lane, 0);
    Quad6 Jq = load_J(Jw, 0, g);
#pragma unroll 1
    for (int step = 0; step < n_steps; ++step) {
        const int hs = step / R_ITERS;                      // half-sweep index in this launch
        const int colour = hs & 1;
        const uint64_t sweep = A.sweep0 + (uint64_t)(hs >> 1);
        const uint32_t time = 2u * (uint32_t)sweep + (uint32_t)colour;
        // prefetch the couplings of the next step
        Geo32 gn = g;
        Quad6 Jn = Jq;
        if (step + 1 < n_steps) {
            const int cn = ((step + 1) / R_ITERS) & 1;
            gn = geo_of(task_of(step + 1), lane, cn);
            Jn = load_J(Jw, cn, gn);
        }
        uint4 *Sa = S4 + colour * RQ;
        const uint4 *So = S4 + (1 - colour) * RQ;
        const uint4 r4 = philox_rk8((uint32_t)g.q, time, wglob, c3, A.rk);
        const bool energy = A.want_energy && hs == 2 * A.n_sweeps - 1;
        if (energy) {
            if (g.p) quad_update<1, true>(Sa, So, g, Jq, r4, K, amask, A.one, A.mone, lane, accU, accM);
            else     quad_update<0, true>(Sa, So, g, Jq, r4, K, amask, A.one, A.mone, lane, accU, accM);
        } else {
            if (g.p) quad_update<1, false>(Sa, So, g, Jq, r4, K, amask, A.one, A.mone, lane, accU, accM);
            else     quad_update<0, false>(Sa, So, g, Jq, r4, K, amask, A.one, A.mone, lane, accU, accM);
        }
        g = gn;
        Jq = Jn;
        if (step % R_ITERS == R_ITERS - 1) __syncthreads();
    }

    if (A.want_energy) {
        const uint32_t totU = bs_warp_total(accU, 8, lane);
        const uint32_t totM = bs_warp_total(accM, 7, lane);
        atomicAdd(&sUM[lane], (int)totU);
        atomicAdd(&sUM[32 + lane], (int)totM);
        __syncthreads();
        if (tid < 32) {
            const size_t o = ((size_t)(w * 32 + tid) * d.R + a) * d.NT + t;
            A.U[o] = (int64_t)sUM[tid];
            A.M[o] = 2 * sUM[32 + tid] - RN;
        }
    }

    // ---- write back
#pragma unroll 8
    for (int i = 0; i < 2 * RQ / R_THREADS; ++i) gS[i * R_THREADS + tid] = S4[i * R_THREADS + tid];
}

constexpr size_t RES32_SMEM = (size_t)RN * 4 + 64 * 4;

}  // namespace

bool res32_supported(const sg_ctx *c)
{
    const Dims &d = c->d;
    return c->kind == SG_PMJ && d.fast_accept && d.L == 32;
}

// n_sweeps consecutive sweeps from global sweep index sweep0; want_energy: also write U, M of the final
// state (fresh energies for the exchange step).  Returns kernels launched (1) or -1.
int launch_res32_pmj(sg_ctx *c, uint64_t sweep0, int n_sweeps, bool want_energy)
{
    static bool configured = false;
    if (!configured) {
        if (cudaFuncSetAttribute(k_res32_pmj, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RES32_SMEM) != cudaSuccess)
            return -1;
        // smallest shared-memory configuration that holds the system: the rest of the 228 KB stays L1
        // and keeps the coupling lines read by the previous half sweep
        cudaFuncSetAttribute(k_res32_pmj, cudaFuncAttributePreferredSharedMemoryCarveout, 58);
        configured = true;
    }
    const Dims &d = c->d;
    Res32Args A;
    A.d = d;
    A.spins = c->spins;
    A.J = c->J;
    A.tab = c->tab;
    A.U = c->U;
    A.M = c->M;
    for (int r = 0; r < 10; ++r) {
        A.rk[2 * r] = d.k0 + (uint32_t)r * 0x9E3779B9u;
        A.rk[2 * r + 1] = d.k1 + (uint32_t)r * 0xBB67AE85u;
    }
    A.sweep0 = sweep0;
    A.n_sweeps = n_sweeps;
    A.want_energy = want_energy ? 1 : 0;
    A.one = 1u;
    A.mone = 0xffffffffu;
    k_res32_pmj<<<d.W * d.R * d.NT, R_THREADS, RES32_SMEM, c->stream>>>(A);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace sg
