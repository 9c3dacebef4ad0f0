// sg_gladder.cu — shared-memory-resident ladder kernel for the Gaussian fp32 path (BASELINE.json config 4).
//
// One CTA owns one (sample s, replica a) ladder: its NT systems (one byte per spin), the sample's fp32
// couplings (3 N floats, shared by all NT systems) and the dexp32 table stay in shared memory for all sweeps
// of a launch, with the exchange step fused in — global memory is touched once per launch instead of twice
// per sweep.  A thread owns one quad (4 consecutive same-colour sites = one Philox call, R6) for the systems
// t = g, g+G, ...; the 24 coupling values of its quad live in registers across those systems.
//
// Arithmetic (R13, R14) is the one of k_sweep_gauss / k_energy_gauss / k_pt_decide_gauss, operation for
// operation: hl = 0 + (+x) + (-x) + (+y) + (-y) + (+z) + (-z) + h in fp32 with separately rounded adds,
// S J applied as a sign-bit flip (exact), dE = +-2 hl, threshold dexp32(beta_f dE); fixed-point int64 energy.
#include "sg_accept.cuh"
#include "sg_device.cuh"
#include "sg_internal.h"

#include <algorithm>

namespace sg {

struct GLadderArgs {
    Dims d;
    int8_t *spins;
    const float *Jg;
    const SlotTab *tab;
    const float *exp32_tab;   // [1441]
    const double *exp64_tab;  // dexp64 table (R12)
    double h;
    float hf;
    uint32_t rk[20];
    uint32_t sweep0;
    int n_sweeps;
    int G;
    int pt_every;
    uint64_t exchange0;
    int64_t *U;               // [S][R][NT]: the kernel's own E_fix, M after the last exchange of the launch (post-swap)
    int32_t *M;
    unsigned long long *pt_acc;   // [NT] accepted swaps per lower slot of the pair
};

namespace {

constexpr int EXP32_N = 1441, EXP32_PAD = 1444;

// sign bit (as a float sign) of byte e of a word of +-1 bytes
__device__ __forceinline__ uint32_t sgn_of(uint32_t w, int e) { return (w << (24 - 8 * e)) & 0x80000000u; }

__device__ __forceinline__ float flip_sign(float J, uint32_t sign) { return __uint_as_float(__float_as_uint(J) ^ sign); }

template <int L>
__global__ void __launch_bounds__(512, 1) k_gladder(const __grid_constant__ GLadderArgs A)
{
    constexpr int Lh = L / 2, N = L * L * L, H = N / 2, Q = H / 4, QR = Lh / 4;
    static_assert(Lh % 4 == 0, "rows must be whole quads");
    extern __shared__ __align__(16) unsigned char sm[];
    const Dims &d = A.d;
    const int NT = d.NT;
    int8_t *S = reinterpret_cast<int8_t *>(sm);                               // [NT][2][H]
    float *Jsm = reinterpret_cast<float *>(sm + (size_t)NT * N);              // [2][3][H]
    float *etab = Jsm + 3 * N;                                                // [EXP32_PAD]
    float *betaf = etab + EXP32_PAD;                                          // [NT]
    long long *Efix = reinterpret_cast<long long *>(betaf + ((NT + 3) & ~3)); // [NT]
    int *Msum = reinterpret_cast<int *>(Efix + NT);                           // [NT]
    int *flags = Msum + NT;                                                   // [NT / 2 + 1]
    int *accs = flags + (NT / 2 + 1);                                         // [NT]

    const int s = blockIdx.x / d.R, a = blockIdx.x % d.R;
    const int tid = threadIdx.x, nthr = blockDim.x;
    int8_t *gS = A.spins + ((size_t)(s * d.R + a) * NT) * N;
    const float *gJ = A.Jg + (size_t)s * 3 * N;

    {
        const uint4 *src = reinterpret_cast<const uint4 *>(gS);
        uint4 *dst = reinterpret_cast<uint4 *>(S);
        for (int i = tid; i < NT * N / 16; i += nthr) dst[i] = src[i];
        const uint4 *js = reinterpret_cast<const uint4 *>(gJ);
        uint4 *jd = reinterpret_cast<uint4 *>(Jsm);
        for (int i = tid; i < 3 * N / 4; i += nthr) jd[i] = js[i];
        for (int i = tid; i < EXP32_N; i += nthr) etab[i] = A.exp32_tab[i];
        for (int i = tid; i < NT; i += nthr) { betaf[i] = A.tab[i].beta_f; accs[i] = 0; }
    }
    __syncthreads();

    const int q = tid % Q, g = tid / Q;
    const bool active = g < A.G;
    const uint32_t sglob = (uint32_t)(s + d.s_first);
    uint64_t exchange = A.exchange0;
    const uint32_t *S32 = reinterpret_cast<const uint32_t *>(S);

    for (int sw = 0; sw < A.n_sweeps; ++sw) {
#pragma unroll 1
        for (int colour = 0; colour < 2; ++colour) {
            if (active) {
                const uint32_t time = 2u * (A.sweep0 + (uint32_t)sw) + (uint32_t)colour;
                const float *Jown = Jsm + (colour * 3) * H;
                const float *Joth = Jsm + ((1 - colour) * 3) * H;
                const int r = q / QR, kq = q % QR;
                const int y = r % L, z = r / L;
                const int p = (colour + y + z) & 1;
                const int q_yp = (y + 1 == L) ? q - (L - 1) * QR : q + QR;
                const int q_ym = (y == 0) ? q + (L - 1) * QR : q - QR;
                const int q_zp = (z + 1 == L) ? q - (L - 1) * L * QR : q + L * QR;
                const int q_zm = (z == 0) ? q + (L - 1) * L * QR : q - L * QR;
                // the one x-neighbour outside this quad: m+1 of element 3 (p = 1) or m-1 of element 0 (p = 0), periodic in the row
                const int m_out = p ? (4 * kq + 4 == Lh ? 0 : 4 * kq + 4) : (kq == 0 ? Lh - 1 : 4 * kq - 1);
                const int side_idx = r * Lh + m_out;
                float Jxp[4], Jxm[4], Jyp[4], Jym[4], Jzp[4], Jzm[4];
                {
                    const float4 jx = reinterpret_cast<const float4 *>(Jown)[q];
                    const float4 jox = reinterpret_cast<const float4 *>(Joth)[q];
                    const float4 jy = reinterpret_cast<const float4 *>(Jown + H)[q];
                    const float4 joy = reinterpret_cast<const float4 *>(Joth + H)[q_ym];
                    const float4 jz = reinterpret_cast<const float4 *>(Jown + 2 * H)[q];
                    const float4 joz = reinterpret_cast<const float4 *>(Joth + 2 * H)[q_zm];
                    const float jside = Joth[side_idx];
                    Jxp[0] = jx.x; Jxp[1] = jx.y; Jxp[2] = jx.z; Jxp[3] = jx.w;           // bond to +x: own
                    // bond to -x: owned by the -x neighbour = same compact index (p) or index m-1 (!p)
                    Jxm[0] = p ? jox.x : jside; Jxm[1] = p ? jox.y : jox.x; Jxm[2] = p ? jox.z : jox.y; Jxm[3] = p ? jox.w : jox.z;
                    Jyp[0] = jy.x; Jyp[1] = jy.y; Jyp[2] = jy.z; Jyp[3] = jy.w;
                    Jym[0] = joy.x; Jym[1] = joy.y; Jym[2] = joy.z; Jym[3] = joy.w;
                    Jzp[0] = jz.x; Jzp[1] = jz.y; Jzp[2] = jz.z; Jzp[3] = jz.w;
                    Jzm[0] = joz.x; Jzm[1] = joz.y; Jzm[2] = joz.z; Jzm[3] = joz.w;
                }
#pragma unroll 1
                for (int t = g; t < NT; t += A.G) {
                    uint32_t *Sa = reinterpret_cast<uint32_t *>(S + (size_t)t * N + colour * H);
                    const uint32_t *So = S32 + ((size_t)t * N + (1 - colour) * H) / 4;
                    const uint32_t sv = Sa[q];
                    const uint32_t o0 = So[q], oyp = So[q_yp], oym = So[q_ym], ozp = So[q_zp], ozm = So[q_zm];
                    const uint32_t sb = (uint32_t)(uint8_t)S[(size_t)t * N + (1 - colour) * H + side_idx];
                    // +x neighbours: same m (!p) or m+1 (p); -x neighbours: m-1 (!p) or same m (p)
                    const uint32_t wxp = p ? ((o0 >> 8) | (sb << 24)) : o0;
                    const uint32_t wxm = p ? o0 : ((o0 << 8) | sb);
                    const uint4 r4 = philox_rk8((uint32_t)q, time, sglob, ctr3(3, a, t), A.rk);
                    const uint32_t rr[4] = {r4.x, r4.y, r4.z, r4.w};
                    const float bf = betaf[t];
                    uint32_t fl = 0;
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        float hl = 0.0f;
                        hl = __fadd_rn(hl, flip_sign(Jxp[e], sgn_of(wxp, e)));
                        hl = __fadd_rn(hl, flip_sign(Jxm[e], sgn_of(wxm, e)));
                        hl = __fadd_rn(hl, flip_sign(Jyp[e], sgn_of(oyp, e)));
                        hl = __fadd_rn(hl, flip_sign(Jym[e], sgn_of(oym, e)));
                        hl = __fadd_rn(hl, flip_sign(Jzp[e], sgn_of(ozp, e)));
                        hl = __fadd_rn(hl, flip_sign(Jzm[e], sgn_of(ozm, e)));
                        hl = __fadd_rn(hl, A.hf);
                        const float two_hl = __fmul_rn(2.0f, hl);
                        const float dE = flip_sign(two_hl, sgn_of(sv, e));          // S > 0 ? 2 hl : -(2 hl)
                        const bool down = dE <= 0.0f;
                        const uint64_t thr = dexp32(etab, __fmul_rn(bf, down ? 0.0f : dE));
                        const bool flip = down || ((uint64_t)rr[e] < thr);
                        fl |= flip ? (0xFEu << (8 * e)) : 0u;                        // +1 (0x01) <-> -1 (0xFF)
                    }
                    Sa[q] = sv ^ fl;
                }
            }
            __syncthreads();
        }
        // ---- exchange step (R12, R14), all in shared memory
        if (A.pt_every > 0 && ((uint64_t)A.sweep0 + (uint64_t)sw + 1) % (uint64_t)A.pt_every == 0) {
            // Energies (R14): thread (q, g) — the mapping of the sweep — takes the quad q of colour 0 (the six bonds of every
            // colour-0 site cover each bond once) for its systems t = g, g + G, ...  The 24 fixed-point couplings of the quad
            // are converted once and stay in registers; per system the spins come as six words, a bond's contribution is
            // selected by the sign byte of S_i xor S_j (one PRMT), and only D = sum over the DIFFERING bonds is accumulated:
            // E_fix = -sum J S_i S_j = 2 D - sum J.  Exact in int64 in any order.  One warp shuffle reduction and one
            // shared-memory atomic per (warp, system) finish the sums.
            const int lane = tid & 31;
            for (int t = tid; t < NT; t += nthr) { Efix[t] = 0; Msum[t] = 0; }
            __syncthreads();
            if (active) {
                const float *Jown = Jsm, *Joth = Jsm + 3 * H;                          // colour 0
                const int r = q / QR, kq = q % QR;
                const int y = r % L, z = r / L;
                const int p = (y + z) & 1;
                const int q_yp = (y + 1 == L) ? q - (L - 1) * QR : q + QR;
                const int q_ym = (y == 0) ? q + (L - 1) * QR : q - QR;
                const int q_zp = (z + 1 == L) ? q - (L - 1) * L * QR : q + L * QR;
                const int q_zm = (z == 0) ? q + (L - 1) * L * QR : q - L * QR;
                const int m_out = p ? (4 * kq + 4 == Lh ? 0 : 4 * kq + 4) : (kq == 0 ? Lh - 1 : 4 * kq - 1);
                const int side_idx = r * Lh + m_out;
                // -J_fix of the 24 bonds as DOUBLES: |J_fix| < 2^36 and every partial sum of a system stays below 2^53, so the
                // additions below are exact (= the int64 sum in any order, R14).  S_i S_j = -1 flips the sign bit of the
                // addend (one shift + one LOP3 on the high word) and the sum runs on the FP64 pipe, not on the ALU pipe.
                double njf[6][4];                                                      // [+x, -x, +y, -y, +z, -z][element]
                {
                    const float4 jx = reinterpret_cast<const float4 *>(Jown)[q];
                    const float4 jox = reinterpret_cast<const float4 *>(Joth)[q];
                    const float4 jy = reinterpret_cast<const float4 *>(Jown + H)[q];
                    const float4 joy = reinterpret_cast<const float4 *>(Joth + H)[q_ym];
                    const float4 jz = reinterpret_cast<const float4 *>(Jown + 2 * H)[q];
                    const float4 joz = reinterpret_cast<const float4 *>(Joth + 2 * H)[q_zm];
                    const float jside = Joth[side_idx];
                    const float Jv[6][4] = {{jx.x, jx.y, jx.z, jx.w},
                                            {p ? jox.x : jside, p ? jox.y : jox.x, p ? jox.z : jox.y, p ? jox.w : jox.z},
                                            {jy.x, jy.y, jy.z, jy.w}, {joy.x, joy.y, joy.z, joy.w},
                                            {jz.x, jz.y, jz.z, jz.w}, {joz.x, joz.y, joz.z, joz.w}};
#pragma unroll
                    for (int k = 0; k < 6; ++k)
#pragma unroll
                        for (int e = 0; e < 4; ++e)
                            njf[k][e] = -(double)__double2ll_rz(__dmul_rn((double)Jv[k][e], 4294967296.0));
                }
#pragma unroll 1
                for (int t = g; t < NT; t += A.G) {
                    const uint32_t *Sa = S32 + ((size_t)t * N) / 4;                    // colour 0
                    const uint32_t *So = S32 + ((size_t)t * N + H) / 4;
                    const uint32_t sv = Sa[q];
                    const uint32_t o0 = So[q], oyp = So[q_yp], oym = So[q_ym], ozp = So[q_zp], ozm = So[q_zm];
                    const uint32_t sb = (uint32_t)(uint8_t)S[(size_t)t * N + H + side_idx];
                    const uint32_t wxp = p ? ((o0 >> 8) | (sb << 24)) : o0;
                    const uint32_t wxm = p ? o0 : ((o0 << 8) | sb);
                    const uint32_t dw[6] = {sv ^ wxp, sv ^ wxm, sv ^ oyp, sv ^ oym, sv ^ ozp, sv ^ ozm};   // byte sign bit: S_i != S_j
                    double ed[4] = {0.0, 0.0, 0.0, 0.0};                               // four chains (exact, so the order is free)
#pragma unroll
                    for (int k = 0; k < 6; ++k)
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            const uint32_t sgn = sgn_of(dw[k], e);                     // 0x80000000 iff S_i != S_j
                            const double term = __hiloint2double(__double2hiint(njf[k][e]) ^ (int)sgn, __double2loint(njf[k][e]));
                            ed[e] = __dadd_rn(ed[e], term);                            // -J S_i S_j
                        }
                    long long ev = __double2ll_rz(__dadd_rn(__dadd_rn(ed[0], ed[1]), __dadd_rn(ed[2], ed[3])));
                    int mv = __dp4a((int)sv, 0x01010101, __dp4a((int)o0, 0x01010101, 0));
                    // warp totals by integer reductions: |ev| < 2^41 (24 bonds of |J_fix| < 2^36), so ev + 2^41 splits into two
                    // 21-bit chunks whose 32-lane sums fit in 32 bits
                    {
                        const unsigned long long evp = (unsigned long long)(ev + (1ll << 41));
                        const unsigned c0 = __reduce_add_sync(0xffffffffu, (unsigned)(evp & 0x1fffffu));
                        const unsigned c1 = __reduce_add_sync(0xffffffffu, (unsigned)(evp >> 21));
                        ev = (long long)c0 + ((long long)c1 << 21) - (32ll << 41);
                        mv = __reduce_add_sync(0xffffffffu, mv);
                    }
                    if (lane == 0) {
                        atomicAdd(reinterpret_cast<unsigned long long *>(&Efix[t]), (unsigned long long)ev);
                        atomicAdd(&Msum[t], mv);
                    }
                }
            }
            __syncthreads();
            const int e1 = (int)(exchange & 1u);
            const int npairs = (NT - e1) / 2;
            if (tid < npairs) {
                const int t = e1 + 2 * tid;
                const double Et = __dsub_rn(__dmul_rn((double)Efix[t], 0x1p-32), __dmul_rn(A.h, (double)Msum[t]));
                const double Eu = __dsub_rn(__dmul_rn((double)Efix[t + 1], 0x1p-32), __dmul_rn(A.h, (double)Msum[t + 1]));
                const double x = __dmul_rn(__dsub_rn(A.tab[t].beta, A.tab[t + 1].beta), __dsub_rn(Et, Eu));
                const uint4 r = philox_rk8(0u, (uint32_t)exchange, sglob, ctr3(4, a, t), A.rk);
                const int acc = ((x >= 0.0) || ((uint64_t)r.x < dexp64(A.exp64_tab, -x))) ? 1 : 0;
                flags[tid] = acc;
                accs[t] += acc;
            }
            __syncthreads();
            if (sw == A.n_sweeps - 1 && tid < NT) {           // publish the energies, permuted like the configurations
                const int p = tid - e1;
                int src = tid;
                if (p >= 0 && (p >> 1) < npairs && flags[p >> 1]) src = (p & 1) ? tid - 1 : tid + 1;
                const size_t o = ((size_t)s * d.R + a) * NT + tid;
                A.U[o] = (int64_t)Efix[src];
                A.M[o] = Msum[src];
            }
            for (int item = tid; item < npairs * (N / 16); item += nthr) {
                const int pair = item / (N / 16), k = item - pair * (N / 16);
                if (!flags[pair]) continue;
                const int t = e1 + 2 * pair;
                uint4 *X = reinterpret_cast<uint4 *>(S + (size_t)t * N) + k;
                uint4 *Y = reinterpret_cast<uint4 *>(S + (size_t)(t + 1) * N) + k;
                const uint4 xv = *X, yv = *Y;
                *X = yv;
                *Y = xv;
            }
            exchange += 1;
            __syncthreads();
        }
    }

    if (tid < NT && accs[tid]) atomicAdd(&A.pt_acc[tid], (unsigned long long)accs[tid]);
    {
        uint4 *dst = reinterpret_cast<uint4 *>(gS);
        const uint4 *src = reinterpret_cast<const uint4 *>(S);
        for (int i = tid; i < NT * N / 16; i += nthr) dst[i] = src[i];
    }
}

size_t gladder_smem(int L, int NT)
{
    const size_t N = (size_t)L * L * L;
    return (size_t)NT * N + 3 * N * 4 + EXP32_PAD * 4 + (size_t)((NT + 3) & ~3) * 4 + (size_t)NT * 8 + (size_t)NT * 4 +
           (size_t)(NT / 2 + 1) * 4 + (size_t)NT * 4 + 16;
}

template <int L>
cudaError_t launch_g(sg_ctx *c, const GLadderArgs &A, int threads, size_t smem, cudaStream_t st, int grid)
{
    if (attr_needed(c, ATTR_GLADDER + (L == 16))) {
        cudaError_t e = cudaFuncSetAttribute(k_gladder<L>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
        if (e != cudaSuccess) return e;
    }
    k_gladder<L><<<grid, threads, smem, st>>>(A);
    return cudaGetLastError();
}

}  // namespace

bool gladder_supported(const sg_ctx *c)
{
    const Dims &d = c->d;
    if (c->path != SG_PATH_AUTO || c->kind != SG_GAUSS) return false;
    if (d.L != 8 && d.L != 16) return false;
    return (size_t)d.NT * d.N % 16 == 0 && gladder_smem(d.L, d.NT) <= (size_t)227 * 1024;
}

// n_sweeps consecutive sweeps from global sweep index sweep0 with the exchanges that fall due fused in
// (pt_every > 0; first exchange index exchange0).  Returns kernels launched (1) or -1.
int launch_gladder(sg_ctx *c, uint64_t sweep0, int n_sweeps, uint64_t exchange0, int pt_every)
{
    const Dims &d = c->d;
    GLadderArgs A;
    A.d = d;
    A.spins = c->spins8;
    A.Jg = c->Jg;
    A.tab = c->tab;
    A.exp32_tab = c->exp32_tab;
    A.exp64_tab = c->exp64_tab;
    A.h = c->h;
    A.hf = (float)c->h;
    for (int r = 0; r < 10; ++r) {
        A.rk[2 * r] = d.k0 + (uint32_t)r * 0x9E3779B9u;
        A.rk[2 * r + 1] = d.k1 + (uint32_t)r * 0xBB67AE85u;
    }
    A.sweep0 = (uint32_t)sweep0;
    A.n_sweeps = n_sweeps;
    A.pt_every = pt_every;
    A.exchange0 = exchange0;
    A.U = c->U;
    A.M = c->M;
    A.pt_acc = c->pt_acc;
    const int Q = d.N / 8;
    int G = std::max(1, std::min(d.NT, 512 / Q));
    for (int gtry = G; gtry >= 1 && gtry * 2 > G; --gtry)
        if (d.NT % gtry == 0) { G = gtry; break; }
    A.G = G;
    const int threads = (Q * G + 31) / 32 * 32;
    if (threads > 512) return -1;
    const size_t smem = gladder_smem(d.L, d.NT);
    const int grid = d.n_samples * d.R;
    const cudaError_t e = d.L == 8 ? launch_g<8>(c, A, threads, smem, c->stream, grid) : launch_g<16>(c, A, threads, smem, c->stream, grid);
    return e == cudaSuccess ? 1 : -1;
}

}  // namespace sg
