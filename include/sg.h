/*
 * sg.h — C-ABI of libsg_b200: the Monte Carlo hot path of arXiv:1403.4560 on one B200 (sm_100a).
 *
 * What the library computes (citations: PAPER.md:<line> of /root/reference/PAPER.md; R<n> = reading
 * n in DESIGN.md §3, taken where the paper is silent):
 *   - the 3D Edwards-Anderson Hamiltonian  H = -sum_<ij> J_ij S_i S_j - h sum_i S_i  on a periodic
 *     L^3 simple-cubic lattice, J_ij = +-1 equiprobable (Eq. 1) or N(0,1) in fp32
 *     (PAPER.md:120 mention; BASELINE.json config 4);
 *   - checkerboard Metropolis sweeps ("spin flip attempt"; R2-R6) of n_samples disorder
 *     samples x n_replicas replicas x n_temps temperature slots;
 *   - parallel tempering between neighbouring temperatures (R12);
 *   - the replica overlap q(k) = (1/N) sum_j S^a_j S^b_j exp(i k.r_j) (Eq. 2) at k = 0
 *     and 12 small wave vectors (R8) for every replica pair, and running sums
 *     of the moments entering Eqs. 3-6 (R9).
 *
 * Conventions
 *   - every function returns SG_OK (0) or a negative sg_status; nothing is printed, nothing exits;
 *     output arguments are untouched on failure; sg_last_error() gives a description.
 *   - "host ptr" / "device ptr" is stated per argument.  The caller owns every buffer it passes.
 *   - all GPU work is enqueued on the stream given to sg_create; calls that fill HOST buffers
 *     synchronise that stream before returning, the others are asynchronous.
 *   - a context is not thread-safe; one context = one GPU (the current device at sg_create).
 *   - site index i = x + L*(y + L*z); sample index s = 32*w + lane for the packed +-J path;
 *     replica pairs in the order (0,1),(0,2),(0,3),(1,2),(1,3),(2,3).
 */
#ifndef SG_B200_H
#define SG_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sg_ctx sg_ctx; /* opaque */

typedef enum sg_status {
    SG_OK = 0,
    SG_EINVAL = -1,       /* bad argument (see each function) */
    SG_ENOMEM = -2,       /* host or device allocation failed / workspace too small */
    SG_ECUDA = -3,        /* a CUDA call or kernel launch failed; sg_last_error has the CUDA string */
    SG_EUNSUPPORTED = -4, /* valid request outside what the kernels support */
    SG_ESTATE = -5        /* call not valid in the current state */
} sg_status;

/* coupling_kind.  SG_PMJ_TPACK: the same +-J model and the same trajectories as SG_PMJ, simulated in the paper's own
 * packing (R17): the temperature copies of one (sample, replica) are the bits of a word, the
 * lattice lives in shared memory, parallel tempering is a bit permutation.  For few samples and many temperatures;
 * L in {4, 6, 8, 10, 12, 16}, n_temps <= 64 (SG_EUNSUPPORTED otherwise). */
enum { SG_PMJ = 0, SG_GAUSS = 1, SG_PMJ_TPACK = 2 };

#define SG_NK 12   /* non-zero wave vectors per record (R8) */
#define SG_REC 25  /* doubles per (sample, slot, pair) record: q(0), Re q(K0), Im q(K0), ... (R9) */
#define SG_NMOM 66 /* accumulator doubles per (sample, slot) (R9) */

/* Bytes of device workspace sg_create needs for these parameters (0 if they are invalid).
 * The workspace must be 256-byte aligned. */
size_t sg_workspace_bytes(int L, int n_samples, int n_replicas, int n_temps, int coupling_kind);

/* Create a simulation: validates, builds the beta / threshold tables on the host in double (R4),
 * and generates couplings and random initial spins on the device from Philox4x32-10 keyed by
 * `seed` (R5, R6).
 *   out           host ptr, receives the context
 *   L             even, 4 <= L <= 64 (checkerboard needs even L; R3)
 *   h             external field, any finite double
 *   n_samples     >= 1 disorder samples; the +-J path packs 32 per uint32 (idle lanes are ignored)
 *   n_replicas    2 or 4 replicas per (sample, temperature) (R9)
 *   temps         host ptr, n_temps temperatures T > 0, non-decreasing (slot 0 coldest; equal neighbours
 *                 are allowed: every proposed swap between them is accepted); copied
 *   n_temps       1 <= n_temps <= 64
 *   coupling_kind SG_PMJ, SG_GAUSS or SG_PMJ_TPACK
 *   workspace     device ptr, 256-byte aligned, >= sg_workspace_bytes(...) bytes, must outlive the
 *                 context; or NULL: the library cudaMallocs (and frees in sg_destroy)
 *   cuda_stream   a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream) or NULL = default
 * Errors: SG_EINVAL (any violated constraint, null out/temps, misaligned workspace), SG_ENOMEM
 * (workspace too small, allocation failure), SG_ECUDA. */
int sg_create(sg_ctx **out, int L, double h, int n_samples, int n_replicas, const double *temps,
              int n_temps, int coupling_kind, uint64_t seed, void *workspace, size_t workspace_bytes,
              void *cuda_stream);

/* Multi-GPU sharding: declare that local sample 0 is global sample `first_sample`
 * of a larger disorder pool, so that every Philox stream is keyed by the GLOBAL sample / word index
 * and results do not depend on how the pool is split over GPUs.  first_sample >= 0, a multiple of
 * 32 for SG_PMJ and SG_PMJ_TPACK.  Takes effect at the next sg_reset (call both right after sg_create). */
int sg_set_first_sample(sg_ctx *ctx, int64_t first_sample);

/* Regenerate couplings and initial spins from the seed, zero the counters and the accumulators:
 * the state right after sg_create, without reallocating.  Asynchronous. */
int sg_reset(sg_ctx *ctx);

/* n >= 0 full checkerboard Metropolis sweeps of every system, colour 0 then colour 1 (R2, R3),
 * no exchange, no measurement.  Asynchronous.  The global sweep counter must stay below 2^31
 * (the Philox time word is 2 * sweep + colour, R6): SG_EINVAL beyond that (also for sg_run). */
int sg_sweep(sg_ctx *ctx, int n);

/* One parallel-tempering exchange step: pairs (t, t+1) with t = e mod 2 for the e-th call (R12),
 * decided per (sample, replica); accepted pairs trade configurations.  Asynchronous. */
int sg_pt_exchange(sg_ctx *ctx);

/* Measure the overlaps of all replica pairs at every slot (Eq. 2) and add their moments to the
 * device accumulators (R9).
 *   out  host ptr to [n_samples][n_temps][n_pairs][SG_REC] doubles, or NULL (then asynchronous). */
int sg_measure(sg_ctx *ctx, double *out);

/* Fused driver, bit-identical to the primitive sequence (R16):
 *   for s in 1..n_sweeps: sweep; if pt_every>0 and sweeps_done % pt_every == 0: exchange;
 *                                if meas_every>0 and sweeps_done % meas_every == 0: measure(NULL)
 * (sweeps_done = global sweep counter).  Asynchronous.
 * Stream order: with a measurement cadence on the +-J ladder paths (L <= 16) the library runs the sweep launches and the
 * measurements on two streams of its own so that a measurement overlaps the sweeps that follow it (DESIGN.md 5,
 * "Overlapped measurements"); both are joined with the context's stream at entry and at exit, so for the caller sg_run
 * behaves like any other call enqueued on `stream`: work enqueued before it is finished when it starts, and everything it
 * did is finished before work enqueued after it starts. */
int sg_run(sg_ctx *ctx, int n_sweeps, int pt_every, int meas_every);

/* Block until all enqueued work of this context has finished. */
int sg_synchronize(sg_ctx *ctx);

/* Free the context and whatever the library allocated (never the caller's workspace). */
int sg_destroy(sg_ctx *ctx);

/* ---- introspection (canonical unpacked layouts, HOST pointers, synchronous) ---- */

/* out: [n_samples][n_replicas][n_temps][N] int8, values +-1 */
int sg_get_spins(sg_ctx *ctx, int8_t *out);
/* in: same layout; any value > 0 means +1 */
int sg_set_spins(sg_ctx *ctx, const int8_t *in);
/* out: [n_samples][3][N] float; entry (d, i) is the bond i -> i+e_d; +-1.0f for SG_PMJ */
int sg_get_couplings(sg_ctx *ctx, float *out);
/* The same three for the samples [s0, s0+ns) only (buffers sized for ns samples): what the
 * parity tests use at full BASELINE.json sizes.  SG_EINVAL if the range is empty or out of bounds. */
int sg_get_spins_range(sg_ctx *ctx, int s0, int ns, int8_t *out);
int sg_set_spins_range(sg_ctx *ctx, int s0, int ns, const int8_t *in);
int sg_get_couplings_range(sg_ctx *ctx, int s0, int ns, float *out);
/* U: [n_samples][n_replicas][n_temps] int64 — SG_PMJ: number of unsatisfied bonds (E = 2U - 3N - hM);
 * SG_GAUSS: fixed-point E_fix = -sum trunc(J 2^32) S_i S_j (R14).  M: same shape int32, sum of spins.
 * Either pointer may be NULL. */
int sg_get_energies(sg_ctx *ctx, int64_t *U, int32_t *M);
/* out: [n_temps][7][2] uint64 Metropolis thresholds thr[t][n_u][a] in [0, 2^32] (R4) */
int sg_get_thresholds(sg_ctx *ctx, uint64_t *out);
/* out: [n_samples][n_temps][SG_NMOM] doubles (may be NULL); n_meas: measurements so far (may be NULL) */
int sg_get_moments(sg_ctx *ctx, double *out, int64_t *n_meas);
/* global sweep / exchange counters (either may be NULL) */
int sg_get_counters(sg_ctx *ctx, uint64_t *sweeps_done, uint64_t *exchanges_done);
/* Checkpoint / resume: every random draw is keyed by the global sweep / exchange counters, so a run continues
 * on the same Philox streams from (spins, counters[, moment accumulators]).  Save with sg_get_spins, sg_get_counters,
 * sg_get_moments; restore into a context created with the SAME parameters and seed (the couplings come from the seed) with
 * sg_set_spins, sg_set_counters and, if measurements are to continue, sg_set_moments.  The continued run is bit-identical to
 * an uninterrupted one.  Not restored: the parallel-tempering statistics (sg_get_pt_stats) and the diagnostics
 * accumulators (P(q), logarithmic-binning windows), which restart from what the new context holds.
 *   sg_set_counters  sweeps_done < 2^31 (SG_EINVAL beyond)
 *   sg_set_moments   in: HOST ptr, [n_samples][n_temps][SG_NMOM] doubles as written by sg_get_moments; n_meas >= 0.
 *                    Synchronous. */
int sg_set_counters(sg_ctx *ctx, uint64_t sweeps_done, uint64_t exchanges_done);
int sg_set_moments(sg_ctx *ctx, const double *in, int64_t n_meas);
/* number of kernels this context has launched so far (for bench.py's gpu_launches) */
int sg_get_launch_count(sg_ctx *ctx, uint64_t *launches);

/* ---- cross-checks and diagnostics of the exchange step ---- */

/* Kernel-path selection.  SG_PATH_AUTO (default) picks the fastest kernels for the shape (ladders or
 * systems resident in shared memory, exchanges fused in); SG_PATH_GENERIC forces the plain
 * global-memory kernels (one launch per half sweep, separate energy / decision / swap / histogram
 * kernels).  Both paths compute the same trajectory bit for bit; the GPU tests compare them over the
 * whole pool through sg_get_state_hash.  May be changed at any time between calls. */
enum { SG_PATH_AUTO = 0, SG_PATH_GENERIC = 1 };
int sg_set_kernel_path(sg_ctx *ctx, int path);

/* One 64-bit hash per system (spin configuration of one packed word / sample, replica, slot):
 * the sum over the system's 32-bit words of mix64(index, word) — independent of the order in which
 * the words are visited.  out: HOST ptr, [n_words][n_replicas][n_temps] with n_words =
 * ceil(n_samples / 32) for SG_PMJ (all 32 lanes of a word, idle lanes included) and n_samples for
 * SG_GAUSS.  Synchronous. */
int sg_get_state_hash(sg_ctx *ctx, uint64_t *out);

/* sg_get_state_hash for callers that cannot allocate device memory.  Same hashes, same layout of `out` (HOST ptr), same
 * synchronous behaviour, but the per-system hashes are staged in one fixed 512 KiB array that is part of the library image
 * (a file-scope __device__ array in csrc/sg_noalloc.cu) instead of a buffer that grows with the pool.  The call and
 * everything under it make no cudaMalloc / cudaFree / cudaMallocAsync call and create no stream or event, so it is safe
 * where those are off limits: inside a host program that has given all device memory to its own pool allocator (a raw
 * cudaMalloc would fail or eat into that pool), in a hook that fires inside a running simulation loop (cudaMalloc and
 * cudaFree stall every stream of the device), or for a caller that was handed a context built on somebody else's
 * workspace and has no allocator at all.  (Create such a context with a caller-owned `workspace`; sg_create with
 * workspace = NULL does allocate.)
 *   limit     n_words * n_replicas * n_temps <= SG_NOALLOC_MAX_SYSTEMS (n_words as for sg_get_state_hash); beyond it
 *             SG_EINVAL, nothing is launched, `out` is untouched and sg_last_error names the limit
 *   cost      the array takes 512 KiB on every GPU that loads this library, until the process exits
 *   first use the first call on each device looks the array's device address up (cudaGetSymbolAddress; this also makes
 *             the runtime load the library's device code there).  Make that first call with the context's device current,
 *             like every other call, and before starting any stream capture; later calls only launch, copy and wait
 *   sharing   all calls on one GPU use the same array and it keeps the previous call's contents.  Nothing needs
 *             clearing (a call reads back only the entries it has just written), but two calls whose GPU work may
 *             overlap, e.g. two contexts driven from two host threads, race on it: serialise them. */
#define SG_NOALLOC_MAX_SYSTEMS 65536
int sg_get_state_hash_noalloc(sg_ctx *ctx, uint64_t *out);

/* The energies the sweep / exchange kernels computed for themselves (what the swap decisions of R12
 * actually used), permuted like the configurations by the exchanges since: same layout as
 * sg_get_energies, which always recounts with a separate kernel.  SG_ESTATE if the kernels' own
 * values are not up to date with the current state (the last operation was a sweep without a
 * following exchange, sg_set_spins, sg_reset). */
int sg_get_energies_cached(sg_ctx *ctx, int64_t *U, int32_t *M);

/* Parallel-tempering statistics since sg_create / sg_reset, per adjacent slot pair (t, t+1),
 * t = 0 .. n_temps-2, summed over samples and replicas: swaps proposed and accepted (R12).
 * HOST ptrs to n_temps-1 values each; either may be NULL.  Synchronous. */
int sg_get_pt_stats(sg_ctx *ctx, uint64_t *proposed, uint64_t *accepted);

/* ---- diagnostics: device-side accumulators, switched on per context ---- */

/* Overlap distribution P(q): from now on every measurement also counts, per (sample, slot), the
 * overlap of every replica pair in a histogram of n_bins bins, 1 <= n_bins <= N + 1.  The integer overlap
 * Q = sum_j S^a_j S^b_j = N q_ab(0) takes N + 1 values; with `agree` = (Q + N) / 2 agreeing sites the bin is
 * floor(agree * n_bins / (N + 1)) (n_bins = N + 1: one bin per value).  The library allocates
 * n_samples * n_temps * n_bins uint32 counters (freed by sg_destroy; zeroed by sg_reset).
 * Errors: SG_EINVAL (n_bins out of range), SG_ENOMEM. */
int sg_enable_pq(sg_ctx *ctx, int n_bins);
/* out: HOST ptr, [n_samples][n_temps][n_bins] uint32.  SG_ESTATE if sg_enable_pq was not called.  Synchronous. */
int sg_get_pq(sg_ctx *ctx, uint32_t *out);

/* Logarithmic-binning equilibration test (Fig. 5 caption): from now on a measurement taken when the
 * global sweep counter is s >= 1 also adds its moments (R9) to the accumulators of window
 * k = min(floor(log2 s), n_windows - 1), i.e. s in [2^k, 2^(k+1)).  1 <= n_windows <= 40.  The library allocates
 * n_windows * n_samples * n_temps * SG_NMOM doubles (freed by sg_destroy; zeroed by sg_reset). */
int sg_enable_log_binning(sg_ctx *ctx, int n_windows);
/* Window k: out HOST ptr [n_samples][n_temps][SG_NMOM] (may be NULL), n_meas = measurements that fell into the window
 * (may be NULL).  SG_ESTATE if not enabled, SG_EINVAL if k is out of range.  Synchronous. */
int sg_get_window_moments(sg_ctx *ctx, int k, double *out, int64_t *n_meas);

/* Which Metropolis comparison the +-J sweep kernels of this context run (it follows from h and the temperatures, DESIGN.md
 * section 5), so that a benchmark can count the arithmetic of the code that actually ran:
 *   SG_ACCEPT_BINARY_SEARCH  h != 0, |h| <= 1: three threshold compares per word-site (26 ALU-pipe lane-ops per word-site)
 *   SG_ACCEPT_CARRY_CHAIN    h == 0: seven compares (30)
 *   SG_ACCEPT_GENERAL        |h| > 1 or a non-monotone table: 14-mask select (no op-count model)
 * SG_EUNSUPPORTED for SG_GAUSS. */
enum { SG_ACCEPT_GENERAL = 0, SG_ACCEPT_CARRY_CHAIN = 1, SG_ACCEPT_BINARY_SEARCH = 2 };
int sg_get_accept_variant(sg_ctx *ctx, int *variant);

/* Fault injection for tests of the error paths: the `countdown`-th resident-ladder launch that sg_run would enqueue from
 * now on (L <= 16 paths) is not enqueued and sg_run returns SG_ECUDA instead; countdown = 0 disarms.  Everything enqueued
 * before it is complete and counted: the context stays usable and a further sg_run continues the same trajectory. */
int sg_debug_fail_launch(sg_ctx *ctx, int countdown);

/* Description of the last error of this context (or of the last failed sg_create if ctx is NULL).
 * The string is owned by the library and valid until the next call on the same context. */
const char *sg_last_error(sg_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* SG_B200_H */
