// sg_internal.h — host-side context and kernel-launcher declarations of libsg_b200 (not installed).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/sg.h"

namespace sg {

constexpr int MAX_NT = 64;
constexpr int N_HIST = 9;   // plane histograms per (sample, slot, pair): x, y, z, x+y, x-y, x+z, x-z, y+z, y-z

// Geometry and keys handed to kernels by value.
struct Dims {
    int L, Lh, N, H;          // L, L/2, L^3, N/2 (sites per colour)
    int R, NT, P;             // replicas, temperature slots, replica pairs
    int W;                    // packed words (PMJ) — ceil(n_samples/32); for GAUSS: n_samples
    int n_samples;
    int s_first;              // global index of local sample 0 (multi-GPU sharding; multiple of 32 for PMJ)
    uint32_t k0, k1;          // Philox key = (seed lo, seed hi)
    uint32_t neg_h;           // 1 if h < 0 (field alignment a = ~s)
    int fast_accept;          // |h| <= 1 and threshold table monotone: comparator path
    int bs_accept;            // fast_accept and every threshold of the codes c <= 6 is < 2^32 (h != 0): binary-search compare
};

// Where a measurement kernel adds its results (R9 + the diagnostics of SURVEY.md 8f rank 4).
struct MeasOut {
    double *acc;              // [n_samples][NT][SG_NMOM] total accumulators
    double *acc_win;          // the same for the current window of the logarithmic-binning test, or NULL
    uint32_t *pq;             // [n_samples][NT][pq_bins] counts of the integer overlap, or NULL
    int pq_bins;
};

// bin of the overlap histogram for `agree` agreeing sites of N (sg_enable_pq): floor(agree * bins / (N + 1))
__host__ __device__ inline int pq_bin(int agree, int N, int bins) { return (int)(((long long)agree * bins) / ((long long)N + 1)); }

// Per-slot device tables (one struct array in the workspace).
struct SlotTab {
    // PMJ fast path: c64[c] = (uint64)(0 - thr(code c)), code c = 2 n_u + (1 - a), c = 0..6
    uint2 c64[7];
    uint2 pad;
    // general path: c64g[n_u][a]
    uint2 c64g[7][2];
    double beta;
    float beta_f;
    float pad2;
};

}  // namespace sg

struct sg_ctx {
    sg::Dims d;
    int kind;
    double h;
    uint64_t seed;
    cudaStream_t stream;
    cudaStream_t stream2;               // measurements that overlap the next ladder launch (sg_run); created lazily
    cudaStream_t stream_hi;             // the ladder launches of such a run (high priority; joined with `stream` at both ends of sg_run)
    cudaEvent_t ev_join;
    cudaEvent_t ev_state;               // ladder stream: the state a measurement reads is complete
    cudaEvent_t ev_read[2];             // stream2: the last measurement reading buffer b (0: lower address) has finished
    bool read_pending[2];
    std::vector<double> temps, beta;
    std::vector<uint64_t> thr;          // [NT][7][2]
    std::string err;
    uint64_t sweeps, exchanges, launches;
    int64_t n_meas;
    int path;                           // SG_PATH_AUTO / SG_PATH_GENERIC (sg_set_kernel_path)
    bool um_fresh;                      // U, M below are the kernels' own energies of the CURRENT state
    bool pending_exchange;              // L = 32 resident path: exchange `exchanges - 1` is decided and applied by the
                                        // next k_res32_pmj launch on load (or by flush_pending), from U, M below
    int fail_countdown;                 // sg_debug_fail_launch: > 0 = the fail_countdown-th ladder launch of sg_run from now reports a failure
    uint32_t attr_done;                 // bit k: cudaFuncSetAttribute done for kernel family k on this context's device
    // device memory
    void *ws;                           // base of the workspace
    size_t ws_bytes;
    bool own_ws;
    uint32_t *spins;                    // PMJ: [W][R][NT][2][H] colour-compacted words (the CURRENT state)
    uint32_t *spins_alt;                // PMJ, L = 32: second state buffer; k_res32_pmj reads `spins`, writes `spins_alt`, then they swap.
                                        // PMJ, L <= 16: the ladder launches of sg_run do the same when a measurement follows them, so that
                                        // the measurement (on `stream2`) can read one buffer while the next launch fills the other
    uint32_t *J;                        // PMJ: [W][2][3][H]
    uint32_t *tps;                      // SG_PMJ_TPACK: [S][R][NW][2][H] temperature-packed state (sg_tpack.cu)
    uint8_t *J6;                        // SG_PMJ_TPACK: [S][2][H] six bond bits per site
    int tp_state;                       // SG_PMJ_TPACK: 0 = both layouts current, 1 = tps newer, 2 = spins (sample-packed) newer
    uint4 *Jp;                          // PMJ, L = 32: couplings repacked per warp step for k_res32_pmj (else NULL)
    int8_t *spins8;                     // GAUSS: [S][R][NT][2][H] colour-compacted bytes
    float *Jg;                          // GAUSS: [S][2][3][H]
    uint32_t *gbits;                    // GAUSS, L <= 16: [chunk / 32][R][NT][2][H] bit-packed copy of a measurement chunk
    sg::SlotTab *tab;                   // [NT]
    double *exp64_tab;                  // [5761]
    float *exp32_tab;                   // [1441]
    double *twiddle;                    // [2][L] cos, sin (2 pi m / L)
    int64_t *U;                         // [S_pad][R][NT]  (S_pad = 32 W for PMJ)
    int32_t *M;                         // [S_pad][R][NT]
    int64_t *U_alt;                     // L = 32: ping-pong partners of U, M (same reason as spins_alt)
    int32_t *M_alt;
    uint32_t *swapmask;                 // PMJ: [W][R][NT/2]; GAUSS: [S][R][NT/2] (0/1)
    uint64_t *hashes;                   // [W][R][NT] scratch of sg_get_state_hash
    unsigned long long *pt_acc;         // [MAX_NT] accepted swaps per lower slot t of the pair (t, t+1), all samples and replicas
    double *acc;                        // [n_samples][NT][SG_NMOM]
    // diagnostics (library-owned allocations, not part of the workspace)
    uint32_t *pq;                       // [n_samples][NT][pq_bins] or NULL (sg_enable_pq)
    int pq_bins;
    double *acc_win;                    // [n_windows][n_samples][NT][SG_NMOM] or NULL (sg_enable_log_binning)
    int n_windows;
    std::vector<int64_t> n_meas_win;    // measurements per window
    uint16_t *hist;                     // scratch [chunk samples][NT][P][N_HIST][L]
    double *rec;                        // scratch [chunk samples][NT][P][SG_REC]
    int chunk_samples;                  // samples per measurement chunk (multiple of 32)
    int8_t *stage8;                     // staging for get/set spins: [chunk][R][NT][N] bytes
};

namespace sg {

// ---- launchers (each returns the number of kernels it launched; errors via cudaGetLastError) ----
int launch_init_pmj(sg_ctx *c);
int launch_init_gauss(sg_ctx *c);
int launch_sweep_pmj(sg_ctx *c, uint64_t sweep);            // both colours
int launch_sweep_gauss(sg_ctx *c, uint64_t sweep);
bool ladder_supported(const sg_ctx *c);                    // shared-memory-resident ladder kernel usable?
// spins_out: where the launch leaves the state (nullptr = in place)
int launch_ladder_pmj(sg_ctx *c, uint64_t sweep0, int n_sweeps, uint64_t exchange0 = 0, int pt_every = 0, uint32_t *spins_out = nullptr);   // 1 launch (-1 on error)
bool gladder_supported(const sg_ctx *c);                   // Gaussian ladder kernel (L = 8, 16) with fused exchanges
int launch_gladder(sg_ctx *c, uint64_t sweep0, int n_sweeps, uint64_t exchange0 = 0, int pt_every = 0);   // 1 launch (-1 on error)
bool ladder8_supported(const sg_ctx *c);                   // L = 8 kernel with fused parallel tempering
int launch_ladder8_pmj(sg_ctx *c, uint64_t sweep0, uint64_t exchange0, int n_sweeps, int pt_every, uint32_t *spins_out = nullptr);
bool res32_supported(const sg_ctx *c);                     // L = 32: one system resident per SM, couplings streamed from L2
size_t res32_packed_bytes(int W);
int launch_pack_J_res32(sg_ctx *c);                        // J -> Jp
// 1 launch (-1 on error): reads c->spins (+ c->U, c->M if do_exchange: decides exchange `exchange` and applies it while
// loading), writes c->spins_alt (+ c->U_alt, c->M_alt if want_energy); the caller swaps the pointers
int launch_res32_pmj(sg_ctx *c, uint64_t sweep0, int n_sweeps, bool want_energy, bool do_exchange, uint64_t exchange);
int launch_energy_pmj(sg_ctx *c);
int launch_energy_gauss(sg_ctx *c);
int launch_pt_pmj(sg_ctx *c, uint64_t exchange);            // decide + swap of spins and of U, M (energies must be fresh)
int launch_pt_gauss(sg_ctx *c, uint64_t exchange);
int launch_hist_pmj(sg_ctx *c, int s0, int ns);             // samples [s0, s0+ns) -> c->hist
int launch_hist_gauss(sg_ctx *c, int s0, int ns);
int launch_finalize(sg_ctx *c, int s0, int ns, bool want_rec);   // hist -> rec (optional), acc
bool measure_fused_supported(const sg_ctx *c);             // bit-sliced one-launch measurement usable?
// spins -> rec (optional), acc; -1 on error.  spins: the packed state to read (nullptr = c->spins), indexed by GLOBAL word
int launch_measure_pmj(sg_ctx *c, int s0, int ns, bool want_rec, const uint32_t *spins = nullptr);
bool measure_fused_gauss_supported(const sg_ctx *c);       // Gaussian path: measurement through a bit-packed copy of the chunk?
int launch_bits_gauss(sg_ctx *c, int s0, int ns);          // byte spins of samples [s0, s0 + ns) -> c->gbits (32 samples per word)
int launch_unpack_pmj(sg_ctx *c, int s0, int ns);           // spins -> stage8 (canonical bytes)
int launch_pack_pmj(sg_ctx *c, int s0, int ns);             // stage8 -> spins (lanes of [s0, s0+ns))
int launch_unpack_gauss(sg_ctx *c, int s0, int ns);
int launch_pack_gauss(sg_ctx *c, int s0, int ns);
int launch_couplings_pmj(sg_ctx *c, int s0, int ns, float *dev_out);   // -> [ns][3][N] float
int launch_couplings_gauss(sg_ctx *c, int s0, int ns, float *dev_out);
size_t tp_state_bytes(int L, int n_samples, int R, int NT);
bool tp_supported(const sg_ctx *c);                        // SG_PMJ_TPACK resident kernel usable?
int launch_tp_pack_J(sg_ctx *c);                           // J -> J6
int launch_tp_from_std(sg_ctx *c);                         // spins -> tps
int launch_tp_to_std(sg_ctx *c);                           // tps -> spins
int launch_tp_run(sg_ctx *c, uint64_t sweep0, int n_sweeps, uint64_t exchange0, int pt_every);   // 1 launch (-1 on error)
inline bool is_packed(const sg_ctx *c) { return c->kind != SG_GAUSS; }   // sample-packed +-J state in c->spins
int launch_hash(sg_ctx *c, uint64_t *dev_out);             // one 64-bit hash per system -> dev_out
// sg_noalloc.cu: hashes of the current state -> out_host through the library's static scratch array (no allocation)
cudaError_t hash_noalloc(sg_ctx *c, uint64_t *out_host, bool *too_large, int *launches);
sg::MeasOut meas_out(const sg_ctx *c);                     // where the measurement kernels add (window from the sweep counter)

// kernel families for sg_ctx::attr_done
enum { ATTR_LADDER8 = 0, ATTR_LADDER = 1, ATTR_GLADDER = 8, ATTR_RES32 = 10, ATTR_MEASURE = 11, ATTR_MEASURE32 = 18, ATTR_GMEASURE = 19, ATTR_TPACK = 24 };
// true if the attribute still has to be set for family `id` on this context (and marks it done)
inline bool attr_needed(sg_ctx *c, int id)
{
    if (c->attr_done & (1u << id)) return false;
    c->attr_done |= 1u << id;
    return true;
}

}  // namespace sg
