// sg_measure.cu — plane histograms -> overlaps q_ab(0), q_ab(K) (Eq. 2) -> records
// and moment accumulators (R7-R9).  Shared by the packed and the byte path.
#include <type_traits>

#include "sg_device.cuh"
#include "sg_internal.h"

namespace sg {

// R9: the moments of one measurement of (sample s, slot t) from its pair records r[pair][SG_REC], added to the
// accumulators (and to the current logarithmic-binning window, if any)
__device__ __forceinline__ void add_records(const Dims &d, const double (&r)[6][SG_REC], int s, int t, const MeasOut &mo)
{
    double a[SG_NMOM];
    for (int j = 0; j < SG_NMOM; ++j) a[j] = 0.0;
    for (int p = 0; p < d.P; ++p) {
        const double v = r[p][0];
        a[0] += v; a[1] += v * v; a[2] += v * v * v; a[3] += (v * v) * (v * v);
        for (int k = 0; k < SG_NK; ++k) {
            const double re = r[p][1 + 2 * k], im = r[p][2 + 2 * k];
            a[4 + 5 * k + 0] += re;
            a[4 + 5 * k + 1] += im;
            a[4 + 5 * k + 2] += re * re + im * im;
        }
    }
    // pair -> (a, b)
    int pa[6], pb[6];
    {
        int p = 0;
        for (int x = 0; x < d.R; ++x)
            for (int y = x + 1; y < d.R; ++y) { pa[p] = x; pb[p] = y; ++p; }
    }
    for (int p = 0; p < d.P; ++p)
        for (int p2 = p + 1; p2 < d.P; ++p2) {
            const int shared = (pa[p] == pa[p2]) + (pa[p] == pb[p2]) + (pb[p] == pa[p2]) + (pb[p] == pb[p2]);
            const int slot = shared == 1 ? 3 : 4;
            a[slot == 3 ? 64 : 65] += r[p][0] * r[p2][0];
            for (int k = 0; k < SG_NK; ++k)
                a[4 + 5 * k + slot] += r[p][1 + 2 * k] * r[p2][1 + 2 * k] + r[p][2 + 2 * k] * r[p2][2 + 2 * k];
        }
    double *A = mo.acc + ((size_t)s * d.NT + t) * SG_NMOM;
    for (int j = 0; j < SG_NMOM; ++j) A[j] += a[j];
    if (mo.acc_win) {
        double *B = mo.acc_win + ((size_t)s * d.NT + t) * SG_NMOM;
        for (int j = 0; j < SG_NMOM; ++j) B[j] += a[j];
    }
}

// One thread per (sample of the chunk, slot): loops over the replica pairs.
// hist: [ns_pad][NT][P][N_HIST][L] uint16 counts of differing sites per plane
// rec : [ns][NT][P][SG_REC] (scratch, copied to the host by sg_measure when asked)
// acc : [n_samples][NT][SG_NMOM]
__global__ void __launch_bounds__(64)
k_finalize(Dims d, const uint16_t *__restrict__ hist, const double *__restrict__ tw, int s0, int ns,
           double *__restrict__ rec, MeasOut mo)
{
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= ns * d.NT) return;
    const int t = tid % d.NT;
    const int sl = tid / d.NT;
    const int L = d.L;
    const double invN = 1.0 / (double)d.N;
    const double *cosv = tw, *sinv = tw + L;
    // which histogram and which harmonic each K uses: K0-2 axes (x1), K3-5 axes (x2), K6-11 diagonals
    const int khist[SG_NK] = {0, 1, 2, 0, 1, 2, 3, 4, 5, 6, 7, 8};
    const int kmul[SG_NK] = {1, 1, 1, 2, 2, 2, 1, 1, 1, 1, 1, 1};
    double r[6][SG_REC];
    for (int p = 0; p < d.P; ++p) {
        const uint16_t *hp = hist + (((size_t)sl * d.NT + t) * d.P + p) * (size_t)(N_HIST * L);
        int D0 = 0;
        for (int m = 0; m < L; ++m) D0 += hp[m];
        r[p][0] = (double)(d.N - 2 * D0) * invN;
        for (int k = 0; k < SG_NK; ++k) {
            const uint16_t *hh = hp + khist[k] * L;
            double re = 0.0, im = 0.0;
            int idx = 0;
            for (int m = 0; m < L; ++m) {
                const double v = (double)(L * L - 2 * (int)hh[m]);    // sum of S^a S^b over the plane
                re += v * cosv[idx];
                im += v * sinv[idx];
                idx += kmul[k];
                if (idx >= L) idx -= L;
            }
            r[p][1 + 2 * k] = re * invN;
            r[p][2 + 2 * k] = im * invN;
        }
        if (rec) {
            double *ro = rec + (((size_t)sl * d.NT + t) * d.P + p) * SG_REC;
            for (int j = 0; j < SG_REC; ++j) ro[j] = r[p][j];
        }
    }
    const int s = s0 + sl;
    if (s >= d.n_samples) return;
    if (mo.pq)
        for (int p = 0; p < d.P; ++p) {
            const uint16_t *hp = hist + (((size_t)sl * d.NT + t) * d.P + p) * (size_t)(N_HIST * L);
            int D0 = 0;
            for (int m = 0; m < L; ++m) D0 += hp[m];
            atomicAdd(&mo.pq[((size_t)s * d.NT + t) * mo.pq_bins + pq_bin(d.N - D0, d.N, mo.pq_bins)], 1u);
        }
    add_records(d, r, s, t, mo);
}

MeasOut meas_out(const sg_ctx *c)
{
    MeasOut mo;
    mo.acc = c->acc;
    mo.pq = c->pq;
    mo.pq_bins = c->pq_bins;
    mo.acc_win = nullptr;
    if (c->acc_win && c->sweeps >= 1) {            // window floor(log2(sweep counter)), clamped to the last one
        int k = 0;
        while ((c->sweeps >> (k + 1)) != 0) ++k;
        if (k > c->n_windows - 1) k = c->n_windows - 1;
        mo.acc_win = c->acc_win + (size_t)k * c->d.n_samples * c->d.NT * SG_NMOM;
    }
    return mo;
}

int launch_finalize(sg_ctx *c, int s0, int ns, bool want_rec)
{
    const Dims &d = c->d;
    const int n = ns * d.NT;
    k_finalize<<<(unsigned)((n + 63) / 64), 64, 0, c->stream>>>(d, c->hist, c->twiddle, s0, ns,
                                                                    want_rec ? c->rec : nullptr, meas_out(c));
    return 1;
}


// ------------------------------------------------------------------ fused bit-sliced measurement
// k_measure_pmj<L>: one CTA per (packed word w, slot t) does everything of a6 + a7 for the 32
// samples of the word: differing-site words D = S^a xor S^b of every replica pair in canonical
// site order (shared memory) -> one thread per (pair, histogram bin) counts its L^2 words with a
// carry-save adder network (bit-sliced: all 32 samples at once) -> one warp transpose per 4 (or 2)
// bins turns the count planes into per-sample integers -> one thread per (pair, sample) does the
// L-point transforms of R7/R8 in double (same arithmetic as k_finalize) -> one thread per
// (sample, moment) adds into the accumulators of R9.
//
// A bin (histogram hh, value b) is the set of sites whose coordinate_hh equals b; it is walked as
// L "outer" x L "inner" sites: idx = u*su + v*sv + ((ku*u + kb) mod L)*sd  (see bin_geometry).

// carry-save adder: (carry, sum) of three one-bit planes
__device__ __forceinline__ void csa(uint32_t &hi, uint32_t &lo, uint32_t a, uint32_t b, uint32_t c)
{
    lo = xor3(a, b, c);
    hi = maj3(a, b, c);
}

// replica pairs in the order (0,1),(0,2),(0,3),(1,2),(1,3),(2,3) (for R = 2 only pair 0 exists):
// do pairs p and p2 share exactly one replica?
__host__ __device__ constexpr bool pairs_share(int p, int p2)
{
    constexpr int A[6] = {0, 0, 0, 1, 1, 2}, B[6] = {1, 2, 3, 2, 3, 3};
    return (A[p] == A[p2]) + (A[p] == B[p2]) + (B[p] == A[p2]) + (B[p] == B[p2]) == 1;
}

template <int L>
struct MeasureCfg {
    static constexpr int N = L * L * L;
    static constexpr int NB = N_HIST * L;                      // bins per pair
    static constexpr int BPB = (L * L < 256) ? 8 : 16;         // bits per bin after the transpose
    static constexpr int PER = 32 / BPB;                       // bins per transposed word
    static constexpr int NG = (NB + PER - 1) / PER;            // 32-word transpose groups per pair
    static constexpr int HI = BPB - 3;                         // planes above ones/twos/fours
    static constexpr int PLW = NG * 32;                        // plane words per pair
};

struct BinGeom {
    int su, sv, sd, ku, kb;
};

template <int L>
__device__ __forceinline__ BinGeom bin_geometry(int hh, int b)
{
    constexpr int L2 = L * L;
    BinGeom g;
    switch (hh) {
    case 0: g = {L, L2, 1, 0, b}; break;          // x = b;       outer y, inner z
    case 1: g = {1, L2, L, 0, b}; break;          // y = b;       outer x, inner z
    case 2: g = {1, L, L2, 0, b}; break;          // z = b;       outer x, inner y
    case 3: g = {1, L2, L, -1, b}; break;         // x + y = b:   y = b - x; outer x, inner z
    case 4: g = {1, L2, L, 1, -b}; break;         // x - y = b:   y = x - b
    case 5: g = {1, L, L2, -1, b}; break;         // x + z = b:   z = b - x; outer x, inner y
    case 6: g = {1, L, L2, 1, -b}; break;         // x - z = b:   z = x - b
    case 7: g = {L, 1, L2, -1, b}; break;         // y + z = b:   z = b - y; outer y, inner x
    default: g = {L, 1, L2, 1, -b}; break;        // y - z = b:   z = y - b
    }
    return g;
}

// ONEPAIR (L = 32, where the differing-site words of one pair already fill 128 KB of shared memory): one CTA per
// (word, slot, replica pair) runs phases 0-3 for its pair and writes the pair's records to `rec`; k_acc_from_rec then
// adds the moments, which need all pairs of a (sample, slot) together.
template <int L, bool ONEPAIR>
__global__ void __launch_bounds__(ONEPAIR ? 288 : 256)
k_measure_pmj(Dims d, const uint32_t *__restrict__ spins, const double *__restrict__ tw, int w0, int s0,
              double *__restrict__ rec, MeasOut mo)
{
    using C = MeasureCfg<L>;
    constexpr int N = C::N, Lh = L / 2, H = N / 2;
    extern __shared__ __align__(16) unsigned char sm_raw[];
    const int P = ONEPAIR ? 1 : d.P;                       // pairs handled by this CTA
    const int pair0 = ONEPAIR ? (int)(blockIdx.x % (unsigned)d.P) : 0;
    const int bidx = ONEPAIR ? (int)(blockIdx.x / (unsigned)d.P) : (int)blockIdx.x;
    // region A: D words [P][N] during the counting phase, then records [P][SG_REC][32] doubles
    uint32_t *Dsm = reinterpret_cast<uint32_t *>(sm_raw);
    double *REC = reinterpret_cast<double *>(sm_raw);
    const size_t regA = ((size_t)P * N * 4 > (size_t)P * SG_REC * 32 * 8) ? (size_t)P * N * 4 : (size_t)P * SG_REC * 32 * 8;
    uint32_t *PL = reinterpret_cast<uint32_t *>(sm_raw + regA);          // [P][NG*32]
    __shared__ double twsm[2 * L];
    __shared__ int pa[6], pb[6], couples[15], n_couples;      // couples: p | p2 << 4 | shared << 8

    const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarp = nthr >> 5;
    const int t = bidx % d.NT;
    const int w = w0 + bidx / d.NT;
    if (tid == 0) {
        int p = 0;
        for (int a = 0; a < d.R; ++a)
            for (int b = a + 1; b < d.R; ++b) { pa[p] = a; pb[p] = b; ++p; }
        int q = 0;
        for (int p1 = 0; p1 < p; ++p1)
            for (int p2 = p1 + 1; p2 < p; ++p2) {
                const int shared = (pa[p1] == pa[p2]) + (pa[p1] == pb[p2]) + (pb[p1] == pa[p2]) + (pb[p1] == pb[p2]);
                couples[q++] = p1 | (p2 << 4) | (shared << 8);
            }
        n_couples = q;
    }
    if (tid < 2 * L) twsm[tid] = tw[tid];
    __syncthreads();

    // ---- phase 0: D = S^a xor S^b, canonical order (every replica's word is loaded once and used by all its pairs)
    if constexpr (ONEPAIR) {
        const uint32_t *A = spins + (((size_t)w * d.R + pa[pair0]) * d.NT + t) * N;
        const uint32_t *B = spins + (((size_t)w * d.R + pb[pair0]) * d.NT + t) * N;
        for (int k4 = tid; k4 < N / 4; k4 += nthr) {                   // four consecutive compact entries = one row segment
            const uint4 av = reinterpret_cast<const uint4 *>(A)[k4], bv = reinterpret_cast<const uint4 *>(B)[k4];
            const uint32_t dv[4] = {av.x ^ bv.x, av.y ^ bv.y, av.z ^ bv.z, av.w ^ bv.w};
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int k = 4 * k4 + e;
                const int c = k / H, n = k - c * H;
                const int row = n / Lh, m = n - row * Lh;
                const int z = row / L, y = row - z * L;
                Dsm[2 * m + ((c + y + z) & 1) + L * (y + L * z)] = dv[e];
            }
        }
    } else
    for (int k4 = tid; k4 < N / 4; k4 += nthr) {                       // four consecutive compact entries: one 128-bit load per replica
        uint4 sr4[4];
#pragma unroll
        for (int a = 0; a < 4; ++a)
            sr4[a] = a < d.R ? reinterpret_cast<const uint4 *>(spins + (((size_t)w * d.R + a) * d.NT + t) * N)[k4] : make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const int k = 4 * k4 + e;                                      // k = colour * H + n
            const int c = k / H, n = k - c * H;
            const int row = n / Lh, m = n - row * Lh;
            const int z = row / L, y = row - z * L;
            const int x = 2 * m + ((c + y + z) & 1);
            const int site = x + L * (y + L * z);
            uint32_t sr[4];
#pragma unroll
            for (int a = 0; a < 4; ++a) sr[a] = e == 0 ? sr4[a].x : e == 1 ? sr4[a].y : e == 2 ? sr4[a].z : sr4[a].w;
#pragma unroll
            for (int pair = 0; pair < 6; ++pair) {
                constexpr int PA[6] = {0, 0, 0, 1, 1, 2}, PB[6] = {1, 2, 3, 2, 3, 3};
                if (pair < P) Dsm[pair * N + site] = sr[PA[pair]] ^ sr[PB[pair]];
            }
        }
    }
    for (int i = tid; i < P * C::PLW; i += nthr) PL[i] = 0u;
    __syncthreads();

    // ---- phase 1: one thread per (pair, bin): bit-sliced count of its L^2 words.  The items are ordered by the stride of the
    // inner loop (L^2: histograms 0, 1, 3, 4; L: 2, 5, 6; 1: 7, 8), each class padded to whole warps, so that a warp runs ONE
    // instantiation with that stride as a compile-time constant: the loads of the unrolled inner loop need no index arithmetic
    {
        constexpr int L2 = L * L;
        const int n0 = P * 4 * L, n1 = P * 3 * L, n2 = P * 2 * L;          // items per class
        const int p0 = (n0 + 31) & ~31, p1 = (n1 + 31) & ~31, p2 = (n2 + 31) & ~31;
        auto count_bin = [&](auto sv_tag, const int pair, const int hh, const int b) {
            constexpr int SV = decltype(sv_tag)::value;
            const int bin = hh * L + b;
            const BinGeom g = bin_geometry<L>(hh, b);
            const uint32_t *Dp = Dsm + pair * N;
            uint32_t ones = 0, twos = 0, fours = 0, hi[C::HI];
#pragma unroll
            for (int k = 0; k < C::HI; ++k) hi[k] = 0;
            // The bins of one histogram (consecutive threads, b = 0 .. L-1) walk their L^2 sites in the same order, and except
            // for the x histogram their addresses differ by multiples of L words: with the walk as written they would meet in
            // the same shared-memory bank at every step.  Thread b therefore starts the loop whose stride is one word (the x
            // direction) at offset b: the sites counted are the same, the banks of a step are all different.
            const int skew_u = g.su == 1 ? b : 0, skew_v = SV == 1 ? b : 0;
#pragma unroll 1
            for (int uu = 0; uu < L; ++uu) {
                int u = uu + skew_u;
                if (u >= L) u -= L;
                int dd = (g.ku * u + g.kb) % L;
                if (dd < 0) dd += L;
                const uint32_t *base = Dp + u * g.su + dd * g.sd;
#pragma unroll
                for (int v0 = 0; v0 < L; v0 += 8) {
                    uint32_t x[8];
#pragma unroll
                    for (int j = 0; j < 8; ++j) {
                        int v = v0 + j + skew_v;
                        if (v >= L) v -= L;
                        x[j] = (v0 + j < L) ? base[v * SV] : 0u;
                    }
                    uint32_t tA, tB, fA, fB, e;
                    csa(tA, ones, ones, x[0], x[1]);
                    csa(tB, ones, ones, x[2], x[3]);
                    csa(fA, twos, twos, tA, tB);
                    csa(tA, ones, ones, x[4], x[5]);
                    csa(tB, ones, ones, x[6], x[7]);
                    csa(fB, twos, twos, tA, tB);
                    csa(e, fours, fours, fA, fB);
                    // ripple the weight-8 carry into the high planes
#pragma unroll
                    for (int k = 0; k < C::HI; ++k) {
                        const uint32_t hk = hi[k];
                        hi[k] = hk ^ e;
                        e = hk & e;
                    }
                }
            }
            uint32_t *out = PL + pair * C::PLW + (bin / C::PER) * 32 + (bin % C::PER) * C::BPB;
            out[0] = ones;
            out[1] = twos;
            out[2] = fours;
#pragma unroll
            for (int k = 0; k < C::HI; ++k) out[3 + k] = hi[k];
        };
        for (int item = tid; item < p0 + p1 + p2; item += nthr) {         // (the class of an item is warp-uniform)
            if (item < p0) {
                if (item < n0) {
                    constexpr int H4[4] = {0, 1, 3, 4};
                    const int pair = item / (4 * L), rem = item - pair * 4 * L;
                    count_bin(std::integral_constant<int, L2>{}, pair, H4[rem / L], rem % L);
                }
            } else if (item < p0 + p1) {
                const int i1 = item - p0;
                if (i1 < n1) {
                    constexpr int H3[3] = {2, 5, 6};
                    const int pair = i1 / (3 * L), rem = i1 - pair * 3 * L;
                    count_bin(std::integral_constant<int, L>{}, pair, H3[rem / L], rem % L);
                }
            } else {
                const int i2 = item - p0 - p1;
                if (i2 < n2) {
                    const int pair = i2 / (2 * L), rem = i2 - pair * 2 * L;
                    count_bin(std::integral_constant<int, 1>{}, pair, 7 + rem / L, rem % L);
                }
            }
        }
    }
    __syncthreads();

    // ---- phase 2: one warp transpose per group: lane l receives the counts of sample 32 w + l
    for (int item = warp; item < P * C::NG; item += nwarp) {
        uint32_t *grp = PL + item * 32;
        const uint32_t v = transpose32(grp[lane], lane);
        __syncwarp();
        grp[lane] = v;
    }
    __syncthreads();

    // ---- phase 3: one thread per (pair, sample): records (same arithmetic as k_finalize)
    const double invN = 1.0 / (double)N;
    for (int item = tid; item < P * 32; item += nthr) {
        const int pair = item >> 5, l = item & 31;
        const uint32_t *cw = PL + pair * C::PLW + l;
        auto cnt = [&](int bin) -> int {
            const uint32_t wv = cw[(bin / C::PER) * 32];
            return (int)((wv >> ((bin % C::PER) * C::BPB)) & ((1u << C::BPB) - 1u));
        };
        double *r = REC + (size_t)pair * SG_REC * 32 + l;         // r[j * 32]
        // REC aliases Dsm (dead since the barrier after phase 1); PL is a separate region
        // per histogram: counts -> plane sums v[m] = L^2 - 2 cnt (registers), then the harmonics that
        // use it (x, y, z: harmonics 1 and 2 = K0-2, K3-5; diagonals: harmonic 1 = K6-11)
        const double *cosv = twsm, *sinv = twsm + L;
#pragma unroll 1
        for (int hh = 0; hh < N_HIST; ++hh) {
            double v[L];
            int tot = 0;
#pragma unroll
            for (int m = 0; m < L; ++m) {
                const int cm = cnt(hh * L + m);
                tot += cm;
                v[m] = (double)(L * L - 2 * cm);
            }
            if (hh == 0) {
                r[0] = (double)(N - 2 * tot) * invN;
                if (mo.pq && w * 32 + l < d.n_samples)       // overlap histogram: N - tot sites agree
                    atomicAdd(&mo.pq[((size_t)(w * 32 + l) * d.NT + t) * mo.pq_bins + pq_bin(N - tot, N, mo.pq_bins)], 1u);
            }
            // (fused multiply-adds: the records are compared to 1e-12, not bit for bit, and -fmad=false would split them)
            double re = 0.0, im = 0.0;
#pragma unroll
            for (int m = 0; m < L; ++m) {
                re = fma(v[m], cosv[m], re);
                im = fma(v[m], sinv[m], im);
            }
            const int k1 = hh < 3 ? hh : hh + 3;
            r[(1 + 2 * k1) * 32] = re * invN;
            r[(2 + 2 * k1) * 32] = im * invN;
            if (hh < 3) {
                double re2 = 0.0, im2 = 0.0;
#pragma unroll
                for (int m = 0; m < L; ++m) {
                    re2 = fma(v[m], cosv[(2 * m) % L], re2);
                    im2 = fma(v[m], sinv[(2 * m) % L], im2);
                }
                r[(1 + 2 * (hh + 3)) * 32] = re2 * invN;
                r[(2 + 2 * (hh + 3)) * 32] = im2 * invN;
            }
        }
    }
    __syncthreads();

    // ---- optional record output: rec[(s - s0)][t][pair][j]
    if (rec) {
        for (int item = tid; item < 32 * P * SG_REC; item += nthr) {
            const int l = item / (P * SG_REC), rest = item - l * (P * SG_REC);
            const int pair = rest / SG_REC, j = rest - pair * SG_REC;
            const int sl = w * 32 + l - s0;
            rec[(((size_t)sl * d.NT + t) * d.P + pair0 + pair) * SG_REC + j] = REC[((size_t)pair * SG_REC + j) * 32 + l];
        }
    }
    if constexpr (ONEPAIR) return;                         // the moments are added by k_acc_from_rec

    // ---- phase 4: one thread per (moment j, sample l), l fastest: j is warp-uniform (no divergence,
    // conflict-free record reads); the sums are staged in shared memory (OUT aliases the plane words,
    // dead since phase 3) and added to the accumulators in coalesced 528-byte runs.
    double *OUT = reinterpret_cast<double *>(PL);                       // [32][OUT_LD]
    constexpr int OUT_LD = SG_NMOM + 1;
    __syncthreads();
    // item = (block kb, sample l): kb < 12: the five moments of wave vector K_kb; kb = 12: q(0) moments
    for (int item = tid; item < 13 * 32; item += nthr) {
        const int kb = item >> 5, l = item & 31;
        const double *R0 = REC + l;
        double *o = OUT + l * OUT_LD;
        if (kb == 12) {
            double v[6], s1 = 0.0, s2 = 0.0, s3 = 0.0, s4 = 0.0;
#pragma unroll
            for (int p = 0; p < 6; ++p) {
                v[p] = 0.0;
                if (p < P) {
                    v[p] = R0[(p * SG_REC) * 32];
                    const double vv = v[p];
                    s1 += vv; s2 += vv * vv; s3 += vv * vv * vv; s4 += (vv * vv) * (vv * vv);
                }
            }
            double c1 = 0.0, c0 = 0.0;
#pragma unroll
            for (int p = 0; p < 6; ++p)
#pragma unroll
                for (int p2 = p + 1; p2 < 6; ++p2)
                    if (p2 < P) {
                        const double pr = v[p] * v[p2];
                        if (pairs_share(p, p2)) c1 += pr; else c0 += pr;
                    }
            o[0] = s1; o[1] = s2; o[2] = s3; o[3] = s4; o[64] = c1; o[65] = c0;
        } else {
            double re[6], im[6], sr = 0.0, si = 0.0, sa = 0.0;
#pragma unroll
            for (int p = 0; p < 6; ++p) {
                re[p] = im[p] = 0.0;
                if (p < P) {
                    re[p] = R0[(p * SG_REC + 1 + 2 * kb) * 32];
                    im[p] = R0[(p * SG_REC + 2 + 2 * kb) * 32];
                    sr += re[p]; si += im[p]; sa += re[p] * re[p] + im[p] * im[p];
                }
            }
            double c1 = 0.0, c0 = 0.0;
#pragma unroll
            for (int p = 0; p < 6; ++p)
#pragma unroll
                for (int p2 = p + 1; p2 < 6; ++p2)
                    if (p2 < P) {
                        const double pr = re[p] * re[p2] + im[p] * im[p2];
                        if (pairs_share(p, p2)) c1 += pr; else c0 += pr;
                    }
            double *ok = o + 4 + 5 * kb;
            ok[0] = sr; ok[1] = si; ok[2] = sa; ok[3] = c1; ok[4] = c0;
        }
    }
    __syncthreads();
    // one addition per address and launch: the reduction instruction gives the same result as load-add-store without
    // waiting for the load.  A warp takes the samples l = warp, warp + nwarp, ...: 66 consecutive doubles per sample
    // (coalesced), no division in the index
    for (int l = warp; l < 32; l += nwarp) {
        const int s = w * 32 + l;
        if (s >= d.n_samples) continue;
        double *A = mo.acc + ((size_t)s * d.NT + t) * SG_NMOM;
        double *B = mo.acc_win ? mo.acc_win + ((size_t)s * d.NT + t) * SG_NMOM : nullptr;
        const double *src = OUT + l * OUT_LD;
#pragma unroll
        for (int j = lane; j < SG_NMOM; j += 32) {
            const double v = src[j];
            atomicAdd(&A[j], v);
            if (B) atomicAdd(&B[j], v);
        }
    }
}

template <int L>
static size_t measure_smem(int P)
{
    using C = MeasureCfg<L>;
    const size_t a = (size_t)P * C::N * 4, b = (size_t)P * SG_REC * 32 * 8;
    const size_t pl = (size_t)P * C::PLW * 4, out = (size_t)32 * (SG_NMOM + 1) * 8;
    return (a > b ? a : b) + (pl > out ? pl : out);
}

template <int L>
static int launch_measure_L(sg_ctx *c, int s0, int ns, bool want_rec, const uint32_t *spins)
{
    const Dims &d = c->d;
    const size_t smem = measure_smem<L>(d.P);
    if (attr_needed(c, ATTR_MEASURE + L / 2 - 2)) {      // L = 4..16 -> ids 11..17
        if (cudaFuncSetAttribute(k_measure_pmj<L, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)measure_smem<L>(6)) != cudaSuccess)
            return -1;
    }
    const int w0 = s0 >> 5, nw = (ns + 31) >> 5;
    k_measure_pmj<L, false><<<(unsigned)(nw * d.NT), 256, smem, c->stream>>>(d, spins ? spins : c->spins, c->twiddle, w0, s0,
                                                                             want_rec ? c->rec : nullptr, meas_out(c));
    return 1;
}

// one thread per (sample of the chunk, slot): records of all pairs -> moment accumulators
__global__ void __launch_bounds__(128)
k_acc_from_rec(Dims d, const double *__restrict__ rec, int s0, int ns, MeasOut mo)
{
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= ns * d.NT) return;
    const int t = tid % d.NT, sl = tid / d.NT;
    if (s0 + sl >= d.n_samples) return;
    double r[6][SG_REC];
    for (int p = 0; p < d.P; ++p)
        for (int j = 0; j < SG_REC; ++j) r[p][j] = rec[(((size_t)sl * d.NT + t) * d.P + p) * SG_REC + j];
    add_records(d, r, s0 + sl, t, mo);
}

// L = 32: one CTA per (word, slot, pair) + the accumulation kernel (records always go through c->rec)
static int launch_measure_32(sg_ctx *c, int s0, int ns)
{
    const Dims &d = c->d;
    const size_t smem = measure_smem<32>(1);
    if (attr_needed(c, ATTR_MEASURE32)) {
        if (cudaFuncSetAttribute(k_measure_pmj<32, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
            return -1;
    }
    const int w0 = s0 >> 5, nw = (ns + 31) >> 5;
    MeasOut mo = meas_out(c), none = mo;
    none.acc = nullptr;                                   // (unused by the ONEPAIR instantiation; P(q) is counted there)
    none.acc_win = nullptr;
    k_measure_pmj<32, true><<<(unsigned)(nw * d.NT * d.P), 288, smem, c->stream>>>(d, c->spins, c->twiddle, w0, s0, c->rec, none);
    mo.pq = nullptr;
    const int n = nw * 32 * d.NT;
    k_acc_from_rec<<<(unsigned)((n + 127) / 128), 128, 0, c->stream>>>(d, c->rec, s0, nw * 32, mo);
    return 2;
}

bool measure_fused_supported(const sg_ctx *c)
{
    const int L = c->d.L;
    return c->path == SG_PATH_AUTO && is_packed(c) && (L == 4 || L == 6 || L == 8 || L == 10 || L == 12 || L == 16 || L == 32);
}

bool measure_fused_gauss_supported(const sg_ctx *c)
{
    const int L = c->d.L;
    return c->path == SG_PATH_AUTO && c->kind == SG_GAUSS && c->gbits != nullptr &&
           (L == 4 || L == 6 || L == 8 || L == 10 || L == 12 || L == 16);
}

// samples [s0, s0+ns), s0 a multiple of 32: records (optional) and accumulators in one launch
int launch_measure_pmj(sg_ctx *c, int s0, int ns, bool want_rec, const uint32_t *spins)
{
    switch (c->d.L) {
    case 4: return launch_measure_L<4>(c, s0, ns, want_rec, spins);
    case 6: return launch_measure_L<6>(c, s0, ns, want_rec, spins);
    case 8: return launch_measure_L<8>(c, s0, ns, want_rec, spins);
    case 10: return launch_measure_L<10>(c, s0, ns, want_rec, spins);
    case 12: return launch_measure_L<12>(c, s0, ns, want_rec, spins);
    case 16: return launch_measure_L<16>(c, s0, ns, want_rec, spins);
    case 32: return launch_measure_32(c, s0, ns);
    default: return -1;
    }
}

}  // namespace sg
