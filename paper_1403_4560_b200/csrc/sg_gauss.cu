// sg_gauss.cu — one-spin-per-byte fp32 path for Gaussian couplings (BASELINE.json config 4;
// DESIGN.md R13, R14).  Arithmetic order is fixed and every fp op is separately rounded, so the
// spin trajectory is bit-identical to the CPU oracle's.
//
// Layout: spins8 [S][R][NT][2][H] int8 (+-1), colour-compacted like the packed path;
//         Jg     [S][2][3][H] float, Jg[s][c][d][n] = bond (i -> i+e_d) owned by site (c, n).
#include "sg_device.cuh"
#include "sg_internal.h"

namespace sg {

struct NbrG {
    int xp, xm, yp, ym, zp, zm;
};

__device__ __forceinline__ NbrG neighbours_g(const Dims &d, int colour, int n)
{
    const int row = n / d.Lh;
    const int m = n - row * d.Lh;
    const int z = row / d.L;
    const int y = row - z * d.L;
    const int p = (colour + y + z) & 1;
    const int side = row * d.Lh + (p ? (m + 1 == d.Lh ? 0 : m + 1) : (m == 0 ? d.Lh - 1 : m - 1));
    NbrG r;
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

__device__ __forceinline__ void site_to_compact_g(const Dims &d, int i, int &colour, int &n)
{
    const int x = i % d.L;
    const int yz = i / d.L;
    colour = (x + yz % d.L + yz / d.L) & 1;
    n = i >> 1;
}

// ------------------------------------------------------------------------------------ init
// Box-Muller in double from 4 Philox words, rounded once to fp32 (R14).
__global__ void k_init_J_gauss(Dims d, float *__restrict__ Jg)
{
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= (long long)d.n_samples * d.N) return;
    const int i = (int)(tid % d.N);
    const int s = (int)(tid / d.N);
    int c, n;
    site_to_compact_g(d, i, c, n);
    const uint4 o = philox4x32_10((uint32_t)i, 0u, (uint32_t)(s + d.s_first), ctr3(1, 0, 0), d.k0, d.k1);
    const double u0 = __dmul_rn(__dadd_rn((double)o.x, 0.5), 0x1p-32);
    const double u1 = __dmul_rn(__dadd_rn((double)o.y, 0.5), 0x1p-32);
    const double u2 = __dmul_rn(__dadd_rn((double)o.z, 0.5), 0x1p-32);
    const double u3 = __dmul_rn(__dadd_rn((double)o.w, 0.5), 0x1p-32);
    double cs, sn;
    double rho = __dsqrt_rn(__dmul_rn(-2.0, dlog(u0)));
    dsincos2pi(u1, &cs, &sn);
    float *base = Jg + ((size_t)(s * 2 + c) * 3) * d.H + n;
    base[0] = __double2float_rn(__dmul_rn(rho, cs));
    base[d.H] = __double2float_rn(__dmul_rn(rho, sn));
    rho = __dsqrt_rn(__dmul_rn(-2.0, dlog(u2)));
    dsincos2pi(u3, &cs, &sn);
    base[2 * d.H] = __double2float_rn(__dmul_rn(rho, cs));
}

__global__ void k_init_S_gauss(Dims d, int8_t *__restrict__ spins)
{
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = (long long)d.n_samples * d.R * d.NT * d.N;
    if (tid >= total) return;
    const int i = (int)(tid % d.N);
    const long long sys = tid / d.N;
    const int t = (int)(sys % d.NT), a = (int)((sys / d.NT) % d.R), s = (int)(sys / (d.NT * d.R));
    int c, n;
    site_to_compact_g(d, i, c, n);
    const uint4 o = philox4x32_10((uint32_t)i, 0u, (uint32_t)(s + d.s_first), ctr3(2, a, t), d.k0, d.k1);
    spins[((size_t)sys * 2 + c) * d.H + n] = (o.x & 1u) ? 1 : -1;
}

// ----------------------------------------------------------------------------------- sweep
// One thread per (system, quad): 4 bytes of the active colour, one Philox call (R6, R13).
__global__ void __launch_bounds__(256)
k_sweep_gauss(Dims d, int8_t *__restrict__ spins, const float *__restrict__ Jg,
              const SlotTab *__restrict__ tab, const float *__restrict__ exp_tab, float hf,
              uint32_t sweep, int colour)
{
    const int Q = d.H >> 2;
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= (long long)d.n_samples * d.R * d.NT * Q) return;
    const int q = (int)(tid % Q);
    const long long sys = tid / Q;
    const int t = (int)(sys % d.NT), a = (int)((sys / d.NT) % d.R), s = (int)(sys / (d.NT * d.R));
    int8_t *act = spins + ((size_t)sys * 2 + colour) * d.H;
    const int8_t *oth = spins + ((size_t)sys * 2 + (1 - colour)) * d.H;
    const float *Jown = Jg + ((size_t)(s * 2 + colour) * 3) * d.H;
    const float *Joth = Jg + ((size_t)(s * 2 + 1 - colour) * 3) * d.H;
    const int H = d.H;
    const float beta_f = tab[t].beta_f;

    char4 sv = *reinterpret_cast<char4 *>(act + 4 * q);
    const uint4 r4 = philox4x32_10((uint32_t)q, 2u * sweep + (uint32_t)colour, (uint32_t)(s + d.s_first), ctr3(3, a, t), d.k0, d.k1);
    signed char sp[4] = {sv.x, sv.y, sv.z, sv.w};
    const uint32_t r[4] = {r4.x, r4.y, r4.z, r4.w};
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const int n = 4 * q + e;
        const NbrG nb = neighbours_g(d, colour, n);
        float hl = 0.0f, J;
        J = Jown[n];              hl = __fadd_rn(hl, oth[nb.xp] > 0 ? J : -J);
        J = Joth[nb.xm];          hl = __fadd_rn(hl, oth[nb.xm] > 0 ? J : -J);
        J = Jown[H + n];          hl = __fadd_rn(hl, oth[nb.yp] > 0 ? J : -J);
        J = Joth[H + nb.ym];      hl = __fadd_rn(hl, oth[nb.ym] > 0 ? J : -J);
        J = Jown[2 * H + n];      hl = __fadd_rn(hl, oth[nb.zp] > 0 ? J : -J);
        J = Joth[2 * H + nb.zm];  hl = __fadd_rn(hl, oth[nb.zm] > 0 ? J : -J);
        hl = __fadd_rn(hl, hf);
        const float two_hl = __fmul_rn(2.0f, hl);
        const float dE = sp[e] > 0 ? two_hl : -two_hl;
        bool flip;
        if (dE <= 0.0f) flip = true;
        else flip = (uint64_t)r[e] < dexp32(exp_tab, __fmul_rn(beta_f, dE));
        if (flip) sp[e] = (signed char)-sp[e];
    }
    *reinterpret_cast<char4 *>(act + 4 * q) = make_char4(sp[0], sp[1], sp[2], sp[3]);
}

// ---------------------------------------------------------------------------------- energy
// E_fix = -sum_bonds trunc(J 2^32) S_i S_j (exact in int64, order-free; R14), M = sum S.
// One block per system; colour-0 sites cover every bond once.
__global__ void __launch_bounds__(128)
k_energy_gauss(Dims d, const int8_t *__restrict__ spins, const float *__restrict__ Jg,
               int64_t *__restrict__ U, int32_t *__restrict__ M)
{
    __shared__ long long shE[4];
    __shared__ int shM[4];
    const long long sys = blockIdx.x;
    const int s = (int)(sys / (d.NT * d.R));
    const int8_t *s0 = spins + ((size_t)sys * 2) * d.H;
    const int8_t *s1 = s0 + d.H;
    const float *J0 = Jg + ((size_t)(s * 2) * 3) * d.H;
    const float *J1 = Jg + ((size_t)(s * 2 + 1) * 3) * d.H;
    const int H = d.H;
    long long e = 0;
    int m = 0;
    for (int n = threadIdx.x; n < H; n += blockDim.x) {
        const NbrG nb = neighbours_g(d, 0, n);
        const int si = s0[n];
        m += si + s1[n];
        long long acc = 0;
        acc += __double2ll_rz(__dmul_rn((double)J0[n], 4294967296.0)) * (long long)(si * s1[nb.xp]);
        acc += __double2ll_rz(__dmul_rn((double)J1[nb.xm], 4294967296.0)) * (long long)(si * s1[nb.xm]);
        acc += __double2ll_rz(__dmul_rn((double)J0[H + n], 4294967296.0)) * (long long)(si * s1[nb.yp]);
        acc += __double2ll_rz(__dmul_rn((double)J1[H + nb.ym], 4294967296.0)) * (long long)(si * s1[nb.ym]);
        acc += __double2ll_rz(__dmul_rn((double)J0[2 * H + n], 4294967296.0)) * (long long)(si * s1[nb.zp]);
        acc += __double2ll_rz(__dmul_rn((double)J1[2 * H + nb.zm], 4294967296.0)) * (long long)(si * s1[nb.zm]);
        e -= acc;
    }
    for (int o = 16; o; o >>= 1) {
        e += __shfl_xor_sync(0xffffffffu, e, o);
        m += __shfl_xor_sync(0xffffffffu, m, o);
    }
    if ((threadIdx.x & 31) == 0) { shE[threadIdx.x >> 5] = e; shM[threadIdx.x >> 5] = m; }
    __syncthreads();
    if (threadIdx.x == 0) {
        long long E = 0;
        int Mm = 0;
        for (int k = 0; k < (int)(blockDim.x >> 5); ++k) { E += shE[k]; Mm += shM[k]; }
        U[sys] = E;
        M[sys] = Mm;
    }
}

// -------------------------------------------------------------------------------------- PT
__global__ void __launch_bounds__(128)
k_pt_decide_gauss(Dims d, const int64_t *__restrict__ U, const int32_t *__restrict__ M,
                  const SlotTab *__restrict__ tab, const double *__restrict__ exp_tab, double h,
                  uint32_t exchange, int npairs, uint32_t *__restrict__ swapmask,
                  unsigned long long *__restrict__ pt_acc)
{
    const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= (long long)d.n_samples * d.R * npairs) return;
    const int pair = (int)(g % npairs), a = (int)((g / npairs) % d.R), s = (int)(g / (npairs * d.R));
    const int t = (int)(exchange & 1u) + 2 * pair;
    const size_t o = ((size_t)s * d.R + a) * d.NT + t;
    const double Et = __dsub_rn(__dmul_rn((double)U[o], 0x1p-32), __dmul_rn(h, (double)M[o]));
    const double Eu = __dsub_rn(__dmul_rn((double)U[o + 1], 0x1p-32), __dmul_rn(h, (double)M[o + 1]));
    const double x = __dmul_rn(__dsub_rn(tab[t].beta, tab[t + 1].beta), __dsub_rn(Et, Eu));
    const uint4 r = philox4x32_10(0u, exchange, (uint32_t)(s + d.s_first), ctr3(4, a, t), d.k0, d.k1);
    const bool accept = (x >= 0.0) || ((uint64_t)r.x < dexp64(exp_tab, -x));
    swapmask[((size_t)s * d.R + a) * (d.NT / 2) + pair] = accept ? 1u : 0u;
    if (accept) atomicAdd(&pt_acc[t], 1ULL);
}

// One CTA per (sample, replica, pair): leaves at once if the pair does not swap; otherwise trades the two
// configurations and their E_fix, M.  The sample index is gridDim.x (limit 2^31 - 1; y and z stop at 65535).
__global__ void __launch_bounds__(256)
k_pt_swap_gauss(Dims d, int8_t *__restrict__ spins, const uint32_t *__restrict__ swapmask,
                uint32_t exchange, int npairs, int64_t *__restrict__ U, int32_t *__restrict__ M)
{
    const int s = blockIdx.x, a = blockIdx.y, pair = blockIdx.z;
    if (!swapmask[((size_t)s * d.R + a) * (d.NT / 2) + pair]) return;
    const int t = (int)(exchange & 1u) + 2 * pair;
    const size_t sys = ((size_t)s * d.R + a) * d.NT + t;
    uint32_t *A = reinterpret_cast<uint32_t *>(spins + sys * d.N);
    uint32_t *B = reinterpret_cast<uint32_t *>(spins + (sys + 1) * d.N);
    for (int j = threadIdx.x; j < (d.N >> 2); j += blockDim.x) {      // N is a multiple of 8
        const uint32_t x = A[j], y = B[j];
        A[j] = y;
        B[j] = x;
    }
    if (threadIdx.x == 0) {
        const int64_t u = U[sys]; U[sys] = U[sys + 1]; U[sys + 1] = u;
        const int32_t m = M[sys]; M[sys] = M[sys + 1]; M[sys + 1] = m;
    }
}

// ------------------------------------------------------------------------------- measurement
// v1: one warp per (sample, slot, pair); lanes split the (z, y) rows, private shared-memory
// histograms, then a cross-lane sum.  Output format identical to k_hist_pmj.
__global__ void __launch_bounds__(32)
k_hist_gauss(Dims d, const int8_t *__restrict__ spins, int s0, uint16_t *__restrict__ hist)
{
    extern __shared__ uint16_t sh[];            // [N_HIST][L][32]
    const int lane = threadIdx.x;
    const int L = d.L;
    int g = blockIdx.x;
    const int pair = g % d.P;  g /= d.P;
    const int t = g % d.NT;    g /= d.NT;
    const int s = s0 + g;
    int ra = 0, rb = 1;
    {
        int p = 0;
        for (int a = 0; a < d.R; ++a)
            for (int b = a + 1; b < d.R; ++b) {
                if (p == pair) { ra = a; rb = b; }
                ++p;
            }
    }
    const int8_t *A = spins + ((((size_t)s * d.R + ra) * d.NT + t) * 2) * d.H;
    const int8_t *B = spins + ((((size_t)s * d.R + rb) * d.NT + t) * 2) * d.H;
    for (int k = 0; k < N_HIST * L; ++k) sh[k * 32 + lane] = 0;
    for (int row = lane; row < L * L; row += 32) {
        const int z = row / L, y = row - z * L;
        int rowcnt = 0;
        for (int x = 0; x < L; ++x) {
            const int c = (x + y + z) & 1;
            const int idx = c * d.H + row * d.Lh + (x >> 1);
            const int bit = (A[idx] != B[idx]) ? 1 : 0;
            rowcnt += bit;
            int b;
            sh[(0 * L + x) * 32 + lane] += bit;
            b = x + y;      if (b >= L) b -= L;  sh[(3 * L + b) * 32 + lane] += bit;
            b = x - y;      if (b < 0) b += L;   sh[(4 * L + b) * 32 + lane] += bit;
            b = x + z;      if (b >= L) b -= L;  sh[(5 * L + b) * 32 + lane] += bit;
            b = x - z;      if (b < 0) b += L;   sh[(6 * L + b) * 32 + lane] += bit;
        }
        int b;
        sh[(1 * L + y) * 32 + lane] += rowcnt;
        sh[(2 * L + z) * 32 + lane] += rowcnt;
        b = y + z;  if (b >= L) b -= L;  sh[(7 * L + b) * 32 + lane] += rowcnt;
        b = y - z;  if (b < 0) b += L;   sh[(8 * L + b) * 32 + lane] += rowcnt;
    }
    __syncwarp();
    uint16_t *out = hist + (((size_t)(s - s0) * d.NT + t) * d.P + pair) * (size_t)(N_HIST * L);
    for (int k = lane; k < N_HIST * L; k += 32) {
        unsigned tot = 0;
        for (int j = 0; j < 32; ++j) tot += sh[k * 32 + ((j + lane) & 31)];
        out[k] = (uint16_t)tot;
    }
}

// Byte spins of 32 consecutive samples -> one word per site (bit j = sample s0 + 32 wl + j, 1 <-> S = +1), the +-J layout
// [wl][R][NT][2][H].  One warp per 128-byte segment of a system: for each of the 32 samples a coalesced 128-byte load
// (lane l: bytes 4 l .. 4 l + 3), the four sign bits of the lane go to bit j of its four output words.  Samples beyond
// n_samples read as S = -1 (their lanes are never accumulated).
__global__ void __launch_bounds__(128)
k_bits_gauss(Dims d, const int8_t *__restrict__ spins, int s0, int n_words, uint32_t *__restrict__ out)
{
    const int lane = threadIdx.x & 31;
    const int n4 = d.N / 4;                                     // uint32 per system in the byte layout = uint4 per system out
    const int segs = (n4 + 31) / 32;
    const long long warp = (long long)blockIdx.x * 4 + (threadIdx.x >> 5);
    if (warp >= (long long)n_words * d.R * d.NT * segs) return;
    const int seg = (int)(warp % segs);
    const long long sys = warp / segs;                          // (wl * R + a) * NT + t
    const int at = (int)(sys % ((long long)d.R * d.NT));
    const int wl = (int)(sys / ((long long)d.R * d.NT));
    const int k = seg * 32 + lane;
    if (k >= n4) return;
    uint32_t w0 = 0, w1 = 0, w2 = 0, w3 = 0;
#pragma unroll 4
    for (int j = 0; j < 32; ++j) {
        const int s = s0 + 32 * wl + j;
        uint32_t v = 0xffffffffu;
        if (s < d.n_samples) v = reinterpret_cast<const uint32_t *>(spins + ((size_t)s * d.R * d.NT + at) * d.N)[k];
        const uint32_t up = ~v;                                 // sign bit of a byte clear <-> S = +1
        w0 |= ((up >> 7) & 1u) << j;
        w1 |= ((up >> 15) & 1u) << j;
        w2 |= ((up >> 23) & 1u) << j;
        w3 |= (up >> 31) << j;
    }
    reinterpret_cast<uint4 *>(out + (size_t)sys * d.N)[k] = make_uint4(w0, w1, w2, w3);
}

// -------------------------------------------------------------------- pack / unpack / getters
__global__ void k_unpack_gauss(Dims d, const int8_t *__restrict__ spins, int s0, int ns, int8_t *__restrict__ out)
{
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = (long long)ns * d.R * d.NT * d.N;
    if (tid >= total) return;
    const int i = (int)(tid % d.N);
    const long long sys = (long long)s0 * d.R * d.NT + tid / d.N;
    int c, n;
    site_to_compact_g(d, i, c, n);
    out[tid] = spins[((size_t)sys * 2 + c) * d.H + n];
}

__global__ void k_pack_gauss(Dims d, int8_t *__restrict__ spins, int s0, int ns, const int8_t *__restrict__ in)
{
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = (long long)ns * d.R * d.NT * d.N;
    if (tid >= total) return;
    const int i = (int)(tid % d.N);
    const long long sys = (long long)s0 * d.R * d.NT + tid / d.N;
    int c, n;
    site_to_compact_g(d, i, c, n);
    spins[((size_t)sys * 2 + c) * d.H + n] = in[tid] > 0 ? 1 : -1;
}

__global__ void k_couplings_gauss(Dims d, const float *__restrict__ Jg, int s0, int ns, float *__restrict__ out)
{
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = (long long)ns * 3 * d.N;
    if (tid >= total) return;
    const int i = (int)(tid % d.N);
    const int dd = (int)((tid / d.N) % 3);
    const int s = s0 + (int)(tid / (3LL * d.N));
    int c, n;
    site_to_compact_g(d, i, c, n);
    out[tid] = Jg[((size_t)(s * 2 + c) * 3 + dd) * d.H + n];
}

// --------------------------------------------------------------------------------- launchers
static inline unsigned blocks_for(long long n, int per) { return (unsigned)((n + per - 1) / per); }

int launch_init_gauss(sg_ctx *c)
{
    const Dims &d = c->d;
    k_init_J_gauss<<<blocks_for((long long)d.n_samples * d.N, 128), 128, 0, c->stream>>>(d, c->Jg);
    k_init_S_gauss<<<blocks_for((long long)d.n_samples * d.R * d.NT * d.N, 256), 256, 0, c->stream>>>(d, c->spins8);
    return 2;
}

int launch_sweep_gauss(sg_ctx *c, uint64_t sweep)
{
    const Dims &d = c->d;
    const long long n = (long long)d.n_samples * d.R * d.NT * (d.H >> 2);
    for (int colour = 0; colour < 2; ++colour)
        k_sweep_gauss<<<blocks_for(n, 256), 256, 0, c->stream>>>(d, c->spins8, c->Jg, c->tab, c->exp32_tab,
                                                                  (float)c->h, (uint32_t)sweep, colour);
    return 2;
}

int launch_energy_gauss(sg_ctx *c)
{
    const Dims &d = c->d;
    k_energy_gauss<<<(unsigned)((long long)d.n_samples * d.R * d.NT), 128, 0, c->stream>>>(d, c->spins8, c->Jg, c->U, c->M);
    return 1;
}

int launch_pt_gauss(sg_ctx *c, uint64_t exchange)
{
    const Dims &d = c->d;
    const int npairs = (d.NT - (int)(exchange & 1)) / 2;
    if (npairs <= 0) return 0;
    k_pt_decide_gauss<<<blocks_for((long long)d.n_samples * d.R * npairs, 128), 128, 0, c->stream>>>(
        d, c->U, c->M, c->tab, c->exp64_tab, c->h, (uint32_t)exchange, npairs, c->swapmask, c->pt_acc);
    k_pt_swap_gauss<<<dim3(d.n_samples, d.R, npairs), 256, 0, c->stream>>>(d, c->spins8, c->swapmask, (uint32_t)exchange,
                                                                           npairs, c->U, c->M);
    return 2;
}

int launch_hist_gauss(sg_ctx *c, int s0, int ns)
{
    const Dims &d = c->d;
    const size_t sh = (size_t)N_HIST * d.L * 32 * sizeof(uint16_t);
    k_hist_gauss<<<(unsigned)(ns * d.NT * d.P), 32, sh, c->stream>>>(d, c->spins8, s0, c->hist);
    return 1;
}

int launch_bits_gauss(sg_ctx *c, int s0, int ns)
{
    const Dims &d = c->d;
    const int n_words = (ns + 31) / 32;
    const long long warps = (long long)n_words * d.R * d.NT * ((d.N / 4 + 31) / 32);
    k_bits_gauss<<<(unsigned)((warps + 3) / 4), 128, 0, c->stream>>>(d, c->spins8, s0, n_words, c->gbits);
    return 1;
}

int launch_unpack_gauss(sg_ctx *c, int s0, int ns)
{
    const Dims &d = c->d;
    k_unpack_gauss<<<blocks_for((long long)ns * d.R * d.NT * d.N, 256), 256, 0, c->stream>>>(d, c->spins8, s0, ns, c->stage8);
    return 1;
}

int launch_pack_gauss(sg_ctx *c, int s0, int ns)
{
    const Dims &d = c->d;
    k_pack_gauss<<<blocks_for((long long)ns * d.R * d.NT * d.N, 256), 256, 0, c->stream>>>(d, c->spins8, s0, ns, c->stage8);
    return 1;
}

int launch_couplings_gauss(sg_ctx *c, int s0, int ns, float *dev_out)
{
    const Dims &d = c->d;
    k_couplings_gauss<<<blocks_for((long long)ns * 3 * d.N, 256), 256, 0, c->stream>>>(d, c->Jg, s0, ns, dev_out);
    return 1;
}

}  // namespace sg
