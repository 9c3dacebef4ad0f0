// sg_measure.cu — plane histograms -> overlaps q_ab(0), q_ab(K) (Eq. 2) -> records
// and moment accumulators (R7-R9).  Shared by the packed and the byte path.
#include "sg_device.cuh"
#include "sg_internal.h"

namespace sg {

// One thread per (sample of the chunk, slot): loops over the replica pairs.
// hist: [ns_pad][NT][P][N_HIST][L] uint16 counts of differing sites per plane
// rec : [ns][NT][P][SG_REC] (scratch, copied to the host by sg_measure when asked)
// acc : [n_samples][NT][SG_NMOM]
__global__ void __launch_bounds__(64)
k_finalize(Dims d, const uint16_t *__restrict__ hist, const double *__restrict__ tw, int s0, int ns,
           double *__restrict__ rec, double *__restrict__ acc)
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
    double *A = acc + ((size_t)s * d.NT + t) * SG_NMOM;
    double a[SG_NMOM];
    for (int j = 0; j < SG_NMOM; ++j) a[j] = A[j];
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
    for (int j = 0; j < SG_NMOM; ++j) A[j] = a[j];
}

int launch_finalize(sg_ctx *c, int s0, int ns, bool want_rec)
{
    const Dims &d = c->d;
    const int n = ns * d.NT;
    k_finalize<<<(unsigned)((n + 63) / 64), 64, 0, c->stream>>>(d, c->hist, c->twiddle, s0, ns,
                                                                    want_rec ? c->rec : nullptr, c->acc);
    return 1;
}

}  // namespace sg
