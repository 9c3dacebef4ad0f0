// sg_api.cu — the C-ABI of libsg_b200 (include/sg.h): argument validation, workspace layout,
// host-side tables (R4, R12, R13), and the call sequences that drive the kernels.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <new>

#include "sg_internal.h"

using namespace sg;

namespace {

thread_local std::string g_create_err;

constexpr size_t ALIGN = 256;
constexpr size_t SCRATCH_CAP = (size_t)128 << 20;    // per scratch buffer
constexpr int DEXP64_N = 5761, DEXP32_N = 1441;

inline size_t up(size_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }

struct Layout {
    size_t spins, spins_alt, gbits, J, Jp, tps, J6, tab, exp64, exp32, tw, U, M, U_alt, M_alt, swap, pt_acc, hashes, acc, hist, rec, stage, total;
    int chunk_meas, chunk_stage, S_pad;
};

bool valid_args(int L, int n_samples, int R, int NT, int kind)
{
    if (L < 4 || L > 64 || (L & 1)) return false;
    if (n_samples < 1 || n_samples > (1 << 24)) return false;
    if (R != 2 && R != 4) return false;
    if (NT < 1 || NT > MAX_NT) return false;
    if (kind != SG_PMJ && kind != SG_GAUSS && kind != SG_PMJ_TPACK) return false;
    return true;
}

Layout make_layout(int L, int n_samples, int R, int NT, int kind)
{
    Layout lo;
    const size_t N = (size_t)L * L * L;
    const int P = R * (R - 1) / 2;
    const int W = (n_samples + 31) / 32;
    lo.S_pad = kind != SG_GAUSS ? W * 32 : n_samples;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off += up(bytes); return o; };
    lo.tps = lo.J6 = 0;
    if (kind != SG_GAUSS) {
        lo.spins = take((size_t)W * R * NT * N * 4);
        // second state buffer: k_res32_pmj reads one buffer and writes the other; so do the ladder launches of sg_run (L <= 16)
        // that a measurement follows
        lo.spins_alt = (kind == SG_PMJ && (L == 32 || L <= 16)) ? take((size_t)W * R * NT * N * 4) : 0;
        lo.J = take((size_t)W * 3 * N * 4);
        lo.Jp = (kind == SG_PMJ && L == 32) ? take(res32_packed_bytes(W)) : 0;
        if (kind == SG_PMJ_TPACK) {
            lo.tps = take(tp_state_bytes(L, n_samples, R, NT));
            lo.J6 = take((size_t)n_samples * N);
        }
    } else {
        lo.Jp = 0;
        lo.spins_alt = 0;
        lo.spins = take((size_t)n_samples * R * NT * N);
        lo.J = take((size_t)n_samples * 3 * N * 4);
    }
    lo.tab = take(sizeof(SlotTab) * NT);
    lo.exp64 = take(sizeof(double) * DEXP64_N);
    lo.exp32 = take(sizeof(float) * DEXP32_N);
    lo.tw = take(sizeof(double) * 2 * L);
    lo.U = take(sizeof(int64_t) * (size_t)lo.S_pad * R * NT);
    lo.M = take(sizeof(int32_t) * (size_t)lo.S_pad * R * NT);
    lo.U_alt = take(sizeof(int64_t) * (size_t)lo.S_pad * R * NT);
    lo.M_alt = take(sizeof(int32_t) * (size_t)lo.S_pad * R * NT);
    lo.pt_acc = take(sizeof(unsigned long long) * MAX_NT);
    lo.hashes = take(sizeof(uint64_t) * (size_t)(kind != SG_GAUSS ? W : n_samples) * R * NT);
    lo.swap = take(sizeof(uint32_t) * (size_t)lo.S_pad * R * (NT / 2 + 1));
    lo.acc = take(sizeof(double) * (size_t)n_samples * NT * SG_NMOM);
    // measurement scratch, chunked over samples (multiples of 32)
    const size_t hist_per = (size_t)NT * P * N_HIST * L * sizeof(uint16_t);
    const size_t rec_per = (size_t)NT * P * SG_REC * sizeof(double);
    size_t cm = SCRATCH_CAP / std::max(hist_per, rec_per);
    cm = std::max<size_t>(32, cm / 32 * 32);
    cm = std::min<size_t>(cm, (size_t)(n_samples + 31) / 32 * 32);
    lo.chunk_meas = (int)cm;
    lo.hist = take(hist_per * cm);
    lo.rec = take(rec_per * cm);
    // Gaussian path: bit-packed copy of one measurement chunk (32 samples per word, the +-J layout), so that the
    // bit-sliced measurement kernel serves both paths
    lo.gbits = (kind == SG_GAUSS && L <= 16) ? take((cm / 32) * (size_t)R * NT * N * 4) : 0;
    const size_t stage_per = std::max((size_t)R * NT * N, 12 * N);
    size_t cs = std::max<size_t>(1, SCRATCH_CAP / stage_per);
    cs = std::min<size_t>(cs, (size_t)n_samples);
    lo.chunk_stage = (int)cs;
    lo.stage = take(stage_per * cs);
    lo.total = off;
    return lo;
}

int fail(sg_ctx *c, int code, const std::string &msg)
{
    if (c) c->err = msg; else g_create_err = msg;
    return code;
}

int check_cuda(sg_ctx *c, cudaError_t e, const char *what)
{
    if (e == cudaSuccess) return SG_OK;
    return fail(c, SG_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

int check_launch(sg_ctx *c, const char *what)
{
    return check_cuda(c, cudaGetLastError(), what);
}

// host tables -> device (R4, R12, R13)
int upload_tables(sg_ctx *c)
{
    const int NT = c->d.NT;
    const double h = c->h;
    std::vector<SlotTab> tabs(NT);
    c->thr.assign((size_t)NT * 14, 0);
    c->beta.resize(NT);
    bool monotone = fabs(h) <= 1.0;
    for (int t = 0; t < NT; ++t) {
        const double beta = 1.0 / c->temps[t];
        c->beta[t] = beta;
        memset(&tabs[t], 0, sizeof(SlotTab));
        tabs[t].beta = beta;
        tabs[t].beta_f = (float)(1.0 / c->temps[t]);
        for (int nu = 0; nu <= 6; ++nu)
            for (int a = 0; a < 2; ++a) {
                const double dE = (double)(12 - 4 * nu) + (a ? 2.0 * fabs(h) : -(2.0 * fabs(h)));
                uint64_t th;
                if (dE <= 0.0) th = 4294967296ULL;
                else {
                    const double p = floor(exp(-beta * dE) * 4294967296.0);
                    th = p >= 4294967296.0 ? 4294967296ULL : (uint64_t)p;
                }
                c->thr[((size_t)t * 7 + nu) * 2 + a] = th;
                const uint64_t neg = (uint64_t)0 - th;
                tabs[t].c64g[nu][a] = make_uint2((uint32_t)neg, (uint32_t)(neg >> 32));
            }
        // comparator path: code c = 2 n_u + (1 - a); needs thr non-decreasing in c and thr = 2^32 for c >= 7
        uint64_t prev = 0;
        for (int code = 0; code < 14; ++code) {
            const int nu = code >> 1, a = 1 - (code & 1);
            const uint64_t th = c->thr[((size_t)t * 7 + nu) * 2 + a];
            if (th < prev) monotone = false;
            if (code >= 7 && th != 4294967296ULL) monotone = false;
            prev = th;
            if (code < 7) tabs[t].c64[code] = tabs[t].c64g[nu][a];
        }
    }
    c->d.fast_accept = monotone ? 1 : 0;
    bool below = monotone;                                  // binary-search compare (sg_accept.cuh): thr[c <= 6] < 2^32
    for (int t = 0; t < NT && below; ++t)
        for (int code = 0; code < 7; ++code)
            if (c->thr[((size_t)t * 7 + (code >> 1)) * 2 + (1 - (code & 1))] >= 4294967296ULL) below = false;
    c->d.bs_accept = below ? 1 : 0;
    std::vector<double> t64(DEXP64_N);
    std::vector<float> t32(DEXP32_N);
    for (int i = 0; i < DEXP64_N; ++i) t64[i] = exp(-(double)i / 256.0);
    for (int i = 0; i < DEXP32_N; ++i) t32[i] = (float)exp(-(double)i / 64.0);
    const int L = c->d.L;
    std::vector<double> tw(2 * L);
    for (int m = 0; m < L; ++m) {
        const double ph = 2.0 * 3.14159265358979323846 * (double)m / (double)L;
        tw[m] = cos(ph);
        tw[L + m] = sin(ph);
    }
    int rc;
    if ((rc = check_cuda(c, cudaMemcpyAsync(c->tab, tabs.data(), sizeof(SlotTab) * NT, cudaMemcpyHostToDevice, c->stream), "upload tab"))) return rc;
    if ((rc = check_cuda(c, cudaMemcpyAsync(c->exp64_tab, t64.data(), sizeof(double) * DEXP64_N, cudaMemcpyHostToDevice, c->stream), "upload exp64"))) return rc;
    if ((rc = check_cuda(c, cudaMemcpyAsync(c->exp32_tab, t32.data(), sizeof(float) * DEXP32_N, cudaMemcpyHostToDevice, c->stream), "upload exp32"))) return rc;
    if ((rc = check_cuda(c, cudaMemcpyAsync(c->twiddle, tw.data(), sizeof(double) * 2 * L, cudaMemcpyHostToDevice, c->stream), "upload twiddle"))) return rc;
    // the host vectors die at return: the copies above come from pageable memory, which
    // cudaMemcpyAsync stages before returning, so this is safe; synchronise anyway (once per create).
    return check_cuda(c, cudaStreamSynchronize(c->stream), "sync after table upload");
}

int do_reset(sg_ctx *c)
{
    const Dims &d = c->d;
    int rc;
    if ((rc = check_cuda(c, cudaMemsetAsync(c->acc, 0, sizeof(double) * (size_t)d.n_samples * d.NT * SG_NMOM, c->stream), "zero acc"))) return rc;
    if ((rc = check_cuda(c, cudaMemsetAsync(c->pt_acc, 0, sizeof(unsigned long long) * MAX_NT, c->stream), "zero pt counters"))) return rc;
    if (c->pq && (rc = check_cuda(c, cudaMemsetAsync(c->pq, 0, sizeof(uint32_t) * (size_t)d.n_samples * d.NT * c->pq_bins, c->stream), "zero P(q)"))) return rc;
    if (c->acc_win && (rc = check_cuda(c, cudaMemsetAsync(c->acc_win, 0, sizeof(double) * (size_t)c->n_windows * d.n_samples * d.NT * SG_NMOM, c->stream), "zero windows"))) return rc;
    std::fill(c->n_meas_win.begin(), c->n_meas_win.end(), 0);
    c->launches += is_packed(c) ? launch_init_pmj(c) : launch_init_gauss(c);
    if (c->Jp) c->launches += launch_pack_J_res32(c);
    if (c->kind == SG_PMJ_TPACK) {
        c->launches += launch_tp_pack_J(c);
        c->tp_state = 2;                                    // the initial state was generated in the sample-packed layout
    }
    c->sweeps = c->exchanges = 0;
    c->n_meas = 0;
    c->um_fresh = false;
    c->pending_exchange = false;
    return check_launch(c, "init kernels");
}

// The L = 32 resident path leaves the exchange that follows its last sweep to the NEXT launch (decision and
// masked swap happen while that launch loads its system).  Anything else that looks at the state first
// materialises it here: decision kernel from the kernels' own U, M, then the masked swap of spins and U, M.
int flush_pending(sg_ctx *c)
{
    if (c->kind == SG_PMJ_TPACK && c->tp_state == 1) {      // the temperature-packed copy is newer: convert it back
        c->launches += launch_tp_to_std(c);
        c->tp_state = 0;
        return check_launch(c, "layout conversion");
    }
    if (!c->pending_exchange) return SG_OK;
    c->pending_exchange = false;
    c->launches += launch_pt_pmj(c, c->exchanges - 1);
    return check_launch(c, "pending exchange");
}

// one exchange step on the current state; the swap kernels permute U, M with the configurations, so the
// energies stay valid afterwards
int do_exchange(sg_ctx *c)
{
    int rc;
    if ((rc = flush_pending(c))) return rc;
    if (!c->um_fresh) c->launches += is_packed(c) ? launch_energy_pmj(c) : launch_energy_gauss(c);
    c->um_fresh = true;
    c->launches += is_packed(c) ? launch_pt_pmj(c, c->exchanges) : launch_pt_gauss(c, c->exchanges);
    if ((rc = check_launch(c, "pt kernels"))) return rc;    // the exchange counter only moves once both kernels are enqueued
    if (c->kind == SG_PMJ_TPACK) c->tp_state = 2;           // the swap ran on the sample-packed copy
    c->exchanges += 1;
    return SG_OK;
}

int do_measure(sg_ctx *c, double *out)
{
    const Dims &d = c->d;
    {
        const int rc = flush_pending(c);
        if (rc) return rc;
    }
    for (int s0 = 0; s0 < d.n_samples; s0 += c->chunk_samples) {
        const int ns = std::min(c->chunk_samples, d.n_samples - s0);
        if (measure_fused_supported(c)) {
            const int k = launch_measure_pmj(c, s0, ns, out != nullptr);
            if (k < 0) return check_launch(c, "measure kernel") ? SG_ECUDA : fail(c, SG_ECUDA, "measure kernel launch failed");
            c->launches += k;
        } else if (measure_fused_gauss_supported(c)) {
            // Gaussian path: the chunk's spins as bits of 32-sample words, then the same bit-sliced measurement kernel
            c->launches += launch_bits_gauss(c, s0, ns);
            const int k = launch_measure_pmj(c, s0, ns, out != nullptr, c->gbits - (size_t)(s0 >> 5) * d.R * d.NT * d.N);
            if (k < 0) return check_launch(c, "measure kernel") ? SG_ECUDA : fail(c, SG_ECUDA, "measure kernel launch failed");
            c->launches += k;
        } else {
            c->launches += is_packed(c) ? launch_hist_pmj(c, s0, ns) : launch_hist_gauss(c, s0, ns);
            c->launches += launch_finalize(c, s0, ns, out != nullptr);
        }
        int rc = check_launch(c, "measure kernels");
        if (rc) return rc;
        if (out) {
            const size_t per = (size_t)d.NT * d.P * SG_REC;
            rc = check_cuda(c, cudaMemcpyAsync(out + (size_t)s0 * per, c->rec, sizeof(double) * per * ns,
                                               cudaMemcpyDeviceToHost, c->stream), "copy records");
            if (rc) return rc;
            rc = check_cuda(c, cudaStreamSynchronize(c->stream), "sync records");
            if (rc) return rc;
        }
    }
    c->n_meas += 1;
    if (c->acc_win && c->sweeps >= 1) {                  // the window meas_out() selected
        int k = 0;
        while ((c->sweeps >> (k + 1)) != 0) ++k;
        c->n_meas_win[std::min(k, c->n_windows - 1)] += 1;
    }
    return SG_OK;
}

// L = 32 resident kernel: n sweeps; applies the pending exchange on load; if `energy_after`, leaves the
// exchange that follows these sweeps pending (its decision needs the energies this launch writes)
int res32_step(sg_ctx *c, int n, bool energy_after)
{
    const int k = launch_res32_pmj(c, c->sweeps, n, energy_after, c->pending_exchange, c->exchanges - 1);
    if (k < 0) return check_launch(c, "res32 kernel") ? SG_ECUDA : fail(c, SG_ECUDA, "res32 kernel launch failed");
    c->launches += k;
    c->sweeps += n;
    std::swap(c->spins, c->spins_alt);
    c->pending_exchange = false;
    c->um_fresh = energy_after;
    if (energy_after) {
        std::swap(c->U, c->U_alt);
        std::swap(c->M, c->M_alt);
        c->pending_exchange = true;
        c->exchanges += 1;
    }
    return SG_OK;
}

// SG_PMJ_TPACK: n sweeps on the temperature-packed state with the exchanges that fall due fused in
int tp_step(sg_ctx *c, int n, int pt_every)
{
    if (c->tp_state == 2) {
        c->launches += launch_tp_from_std(c);
        c->tp_state = 0;
    }
    const int k = launch_tp_run(c, c->sweeps, n, c->exchanges, pt_every);
    if (k < 0) return check_launch(c, "tpack kernel") ? SG_ECUDA : fail(c, SG_ECUDA, "tpack kernel launch failed");
    c->launches += k;
    if (pt_every > 0) c->exchanges += (c->sweeps + (uint64_t)n) / (uint64_t)pt_every - c->sweeps / (uint64_t)pt_every;
    c->sweeps += n;
    c->um_fresh = pt_every > 0 && c->sweeps % (uint64_t)pt_every == 0;
    c->tp_state = 1;
    return SG_OK;
}

// n consecutive sweeps with nothing in between
int do_sweeps(sg_ctx *c, int n)
{
    if (n <= 0) return SG_OK;
    int rc;
    if (tp_supported(c)) return tp_step(c, n, 0);
    if (res32_supported(c)) return res32_step(c, n, false);
    if ((rc = flush_pending(c))) return rc;
    c->um_fresh = false;
    if (ladder8_supported(c)) {
        const int k = launch_ladder8_pmj(c, c->sweeps, c->exchanges, n, 0);
        if (k < 0) return check_launch(c, "ladder8 kernel") ? SG_ECUDA : fail(c, SG_ECUDA, "ladder8 kernel launch failed");
        c->launches += k;
        c->sweeps += n;
        return SG_OK;
    }
    if (gladder_supported(c)) {
        const int k = launch_gladder(c, c->sweeps, n);
        if (k < 0) return check_launch(c, "gauss ladder kernel") ? SG_ECUDA : fail(c, SG_ECUDA, "gauss ladder kernel launch failed");
        c->launches += k;
        c->sweeps += n;
        return SG_OK;
    }
    if (ladder_supported(c)) {
        const int k = launch_ladder_pmj(c, c->sweeps, n);
        if (k < 0) return check_launch(c, "ladder kernel") ? SG_ECUDA : fail(c, SG_ECUDA, "ladder kernel launch failed");
        c->launches += k;
        c->sweeps += n;
        return SG_OK;
    }
    for (int i = 0; i < n; ++i) {
        c->launches += is_packed(c) ? launch_sweep_pmj(c, c->sweeps) : launch_sweep_gauss(c, c->sweeps);
        c->sweeps += 1;
    }
    if (c->kind == SG_PMJ_TPACK) c->tp_state = 2;
    return SG_OK;
}

bool sweeps_overflow(const sg_ctx *c, int n) { return c->sweeps + (uint64_t)n >= (1ull << 31); }

}  // namespace

extern "C" {

size_t sg_workspace_bytes(int L, int n_samples, int n_replicas, int n_temps, int coupling_kind)
{
    if (!valid_args(L, n_samples, n_replicas, n_temps, coupling_kind)) return 0;
    return make_layout(L, n_samples, n_replicas, n_temps, coupling_kind).total;
}

int sg_create(sg_ctx **out, int L, double h, int n_samples, int n_replicas, const double *temps, int n_temps,
              int coupling_kind, uint64_t seed, void *workspace, size_t workspace_bytes, void *cuda_stream)
{
    if (!out) return fail(nullptr, SG_EINVAL, "sg_create: out is NULL");
    if (!temps) return fail(nullptr, SG_EINVAL, "sg_create: temps is NULL");
    if (!valid_args(L, n_samples, n_replicas, n_temps, coupling_kind))
        return fail(nullptr, SG_EINVAL, "sg_create: need even 4<=L<=64, 1<=n_samples<=2^24, n_replicas in {2,4}, 1<=n_temps<=64, coupling_kind in {0 (SG_PMJ), 1 (SG_GAUSS), 2 (SG_PMJ_TPACK)}");
    if (!(h == h) || fabs(h) > 1e300) return fail(nullptr, SG_EINVAL, "sg_create: h must be finite");
    for (int t = 0; t < n_temps; ++t) {
        if (!(temps[t] > 0.0) || !(temps[t] < 1e308)) return fail(nullptr, SG_EINVAL, "sg_create: temperatures must be finite and > 0");
        if (t && temps[t] < temps[t - 1]) return fail(nullptr, SG_EINVAL, "sg_create: temperatures must be non-decreasing");
    }
    const Layout lo = make_layout(L, n_samples, n_replicas, n_temps, coupling_kind);
    if (workspace) {
        if (((uintptr_t)workspace) % ALIGN) return fail(nullptr, SG_EINVAL, "sg_create: workspace must be 256-byte aligned");
        if (workspace_bytes < lo.total) return fail(nullptr, SG_ENOMEM, "sg_create: workspace smaller than sg_workspace_bytes()");
    }
    sg_ctx *c = new (std::nothrow) sg_ctx();
    if (!c) return fail(nullptr, SG_ENOMEM, "sg_create: host allocation failed");
    c->kind = coupling_kind;
    c->h = h;
    c->seed = seed;
    c->stream = (cudaStream_t)cuda_stream;
    c->temps.assign(temps, temps + n_temps);
    c->sweeps = c->exchanges = c->launches = 0;
    c->n_meas = 0;
    c->path = SG_PATH_AUTO;
    c->pq = nullptr;
    c->pq_bins = 0;
    c->acc_win = nullptr;
    c->n_windows = 0;
    c->um_fresh = false;
    c->pending_exchange = false;
    c->attr_done = 0;
    c->fail_countdown = 0;
    Dims &d = c->d;
    d.L = L; d.Lh = L / 2; d.N = L * L * L; d.H = d.N / 2;
    d.R = n_replicas; d.NT = n_temps; d.P = n_replicas * (n_replicas - 1) / 2;
    d.n_samples = n_samples;
    d.W = coupling_kind != SG_GAUSS ? (n_samples + 31) / 32 : n_samples;
    d.k0 = (uint32_t)seed; d.k1 = (uint32_t)(seed >> 32);
    d.neg_h = h < 0.0 ? 1u : 0u;
    d.fast_accept = 0;
    d.bs_accept = 0;
    d.s_first = 0;
    c->own_ws = workspace == nullptr;
    c->ws_bytes = lo.total;
    if (workspace) c->ws = workspace;
    else {
        cudaError_t e = cudaMalloc(&c->ws, lo.total);
        if (e != cudaSuccess) {
            g_create_err = std::string("sg_create: cudaMalloc: ") + cudaGetErrorString(e);
            delete c;
            return SG_ENOMEM;
        }
    }
    char *b = (char *)c->ws;
    c->spins = (uint32_t *)(b + lo.spins);
    c->spins8 = (int8_t *)(b + lo.spins);
    c->spins_alt = (coupling_kind == SG_PMJ && (L == 32 || L <= 16)) ? (uint32_t *)(b + lo.spins_alt) : nullptr;
    c->stream2 = nullptr;
    c->stream_hi = nullptr;
    c->ev_join = nullptr;
    c->ev_state = nullptr;
    c->ev_read[0] = c->ev_read[1] = nullptr;
    c->read_pending[0] = c->read_pending[1] = false;
    c->gbits = (coupling_kind == SG_GAUSS && L <= 16) ? (uint32_t *)(b + lo.gbits) : nullptr;
    c->J = (uint32_t *)(b + lo.J);
    c->Jg = (float *)(b + lo.J);
    c->Jp = (coupling_kind == SG_PMJ && L == 32) ? (uint4 *)(b + lo.Jp) : nullptr;
    c->tps = coupling_kind == SG_PMJ_TPACK ? (uint32_t *)(b + lo.tps) : nullptr;
    c->J6 = coupling_kind == SG_PMJ_TPACK ? (uint8_t *)(b + lo.J6) : nullptr;
    c->tp_state = 0;
    c->tab = (SlotTab *)(b + lo.tab);
    c->exp64_tab = (double *)(b + lo.exp64);
    c->exp32_tab = (float *)(b + lo.exp32);
    c->twiddle = (double *)(b + lo.tw);
    c->U = (int64_t *)(b + lo.U);
    c->M = (int32_t *)(b + lo.M);
    c->U_alt = (int64_t *)(b + lo.U_alt);
    c->M_alt = (int32_t *)(b + lo.M_alt);
    c->swapmask = (uint32_t *)(b + lo.swap);
    c->pt_acc = (unsigned long long *)(b + lo.pt_acc);
    c->hashes = (uint64_t *)(b + lo.hashes);
    c->acc = (double *)(b + lo.acc);
    c->hist = (uint16_t *)(b + lo.hist);
    c->rec = (double *)(b + lo.rec);
    c->stage8 = (int8_t *)(b + lo.stage);
    c->chunk_samples = lo.chunk_meas;
    int rc = upload_tables(c);
    if (!rc && coupling_kind == SG_PMJ_TPACK && !tp_supported(c))
        rc = fail(c, SG_EUNSUPPORTED, "sg_create: SG_PMJ_TPACK needs L in {4, 6, 8, 10, 12, 16} and a (sample, replica) lattice that fits in shared memory");
    if (!rc) rc = do_reset(c);
    if (rc) {
        g_create_err = c->err;
        if (c->own_ws) cudaFree(c->ws);
        delete c;
        return rc;
    }
    *out = c;
    return SG_OK;
}

int sg_set_first_sample(sg_ctx *c, int64_t first_sample)
{
    if (!c) return SG_EINVAL;
    if (first_sample < 0 || first_sample > 0x7fffffff - c->d.n_samples - 32 || (c->kind != SG_GAUSS && (first_sample & 31)))
        return fail(c, SG_EINVAL, "sg_set_first_sample: need 0 <= first_sample < 2^31, a multiple of 32 for SG_PMJ / SG_PMJ_TPACK");
    c->d.s_first = (int)first_sample;
    return SG_OK;
}

int sg_reset(sg_ctx *c)
{
    if (!c) return SG_EINVAL;
    return do_reset(c);
}

int sg_sweep(sg_ctx *c, int n)
{
    if (!c) return SG_EINVAL;
    if (n < 0) return fail(c, SG_EINVAL, "sg_sweep: n < 0");
    if (sweeps_overflow(c, n)) return fail(c, SG_EINVAL, "sg_sweep: the global sweep counter must stay below 2^31");
    // no flush_pending here: do_sweeps flushes on the paths that need the materialised state; the temperature-packed kernel
    // continues from its own layout and the L = 32 kernel applies a pending exchange while it loads
    const int rc = do_sweeps(c, n);
    if (rc) return rc;
    return check_launch(c, "sweep kernels");
}

int sg_pt_exchange(sg_ctx *c)
{
    if (!c) return SG_EINVAL;
    return do_exchange(c);
}

int sg_measure(sg_ctx *c, double *out)
{
    if (!c) return SG_EINVAL;
    return do_measure(c, out);
}

int sg_run(sg_ctx *c, int n_sweeps, int pt_every, int meas_every)
{
    if (!c) return SG_EINVAL;
    if (n_sweeps < 0 || pt_every < 0 || meas_every < 0) return fail(c, SG_EINVAL, "sg_run: negative argument");
    if (sweeps_overflow(c, n_sweeps)) return fail(c, SG_EINVAL, "sg_run: the global sweep counter must stay below 2^31");
    int left = n_sweeps, rc;
    if (tp_supported(c)) {
        // sweeps and exchanges fused in one launch on the temperature-packed state; launches end at measurements
        while (left > 0) {
            uint64_t run = (uint64_t)left;
            if (meas_every > 0) run = std::min<uint64_t>(run, (uint64_t)meas_every - c->sweeps % (uint64_t)meas_every);
            if ((rc = tp_step(c, (int)run, pt_every))) return rc;
            left -= (int)run;
            if (meas_every > 0 && c->sweeps % (uint64_t)meas_every == 0)
                if ((rc = do_measure(c, nullptr))) return rc;
        }
        return check_launch(c, "run kernels");
    }
    if (ladder8_supported(c) || ladder_supported(c) || gladder_supported(c)) {
        // sweeps and the exchanges between them are fused in one launch; launches end at measurements.
        // +-J: a launch that a measurement follows leaves the state in the SECOND buffer; the measurement then runs on a
        // stream of its own and reads that buffer while the next launch (which reads it too) fills the first one again -
        // measurement CTAs take the SMs and shared memory the ladder CTAs leave free (C3: the last, 46 % full wave).
        const bool overlap = meas_every > 0 && c->kind == SG_PMJ && c->spins_alt && measure_fused_supported(c) &&
                             (ladder8_supported(c) || ladder_supported(c));
        if (overlap && !c->stream2) {
            // the ladder launches of an overlapped run go to a HIGH-priority stream of the library, the measurements to a
            // low-priority one: the block scheduler then places a measurement CTA only where no ladder CTA fits
            // All six objects are created into locals and handed to the context together: a failure half way leaves the
            // context as it was (nothing leaks, the next call tries again) instead of a stream without its events.
            int lo_pri = 0, hi_pri = 0;
            cudaDeviceGetStreamPriorityRange(&lo_pri, &hi_pri);
            cudaStream_t s_hi = nullptr, s_lo = nullptr;
            cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
            cudaError_t e = cudaStreamCreateWithPriority(&s_hi, cudaStreamNonBlocking, hi_pri);
            if (e == cudaSuccess) e = cudaStreamCreateWithPriority(&s_lo, cudaStreamNonBlocking, lo_pri);
            for (int i = 0; i < 4 && e == cudaSuccess; ++i) e = cudaEventCreateWithFlags(&ev[i], cudaEventDisableTiming);
            if (e != cudaSuccess) {
                for (cudaEvent_t x : ev)
                    if (x) cudaEventDestroy(x);
                if (s_lo) cudaStreamDestroy(s_lo);
                if (s_hi) cudaStreamDestroy(s_hi);
                return check_cuda(c, e, "sg_run: streams / events of the overlapped measurements");
            }
            c->stream_hi = s_hi;
            c->stream2 = s_lo;
            c->ev_join = ev[0];
            c->ev_state = ev[1];
            c->ev_read[0] = ev[2];
            c->ev_read[1] = ev[3];
        }
        auto buf_id = [&](const uint32_t *p) { return p == std::min(c->spins, c->spins_alt) ? 0 : 1; };
        // An overlapped measurement is SUBMITTED after the next ladder launch, so that the ladder CTAs are placed first
        // and the measurement CTAs fill what is left; it still sees the buffer and the sweep counter it belongs to.
        bool deferred = false;
        uint32_t *def_buf = nullptr;
        uint64_t def_sweeps = 0;
        auto submit_deferred = [&]() -> int {
            if (!deferred) return SG_OK;
            deferred = false;
            int r = check_cuda(c, cudaStreamWaitEvent(c->stream2, c->ev_state, 0), "wait state");
            if (r) return r;
            uint32_t *cur = c->spins;
            const uint64_t cur_sweeps = c->sweeps;
            c->spins = def_buf;
            c->sweeps = def_sweeps;
            std::swap(c->stream, c->stream2);
            r = do_measure(c, nullptr);
            std::swap(c->stream, c->stream2);
            c->spins = cur;
            c->sweeps = cur_sweeps;
            if (r) return r;
            if ((r = check_cuda(c, cudaEventRecord(c->ev_read[buf_id(def_buf)], c->stream2), "record measurement"))) return r;
            c->read_pending[buf_id(def_buf)] = true;
            return SG_OK;
        };
        cudaStream_t user_stream = c->stream;
        if (overlap) {                                              // the library's streams start where the caller's stream is
            if ((rc = check_cuda(c, cudaEventRecord(c->ev_join, user_stream), "record entry"))) return rc;
            if ((rc = check_cuda(c, cudaStreamWaitEvent(c->stream_hi, c->ev_join, 0), "wait entry"))) return rc;
            c->stream = c->stream_hi;
        }
        auto run_loop = [&]() -> int {
        while (left > 0) {
            uint64_t run = (uint64_t)left;
            if (meas_every > 0) run = std::min<uint64_t>(run, (uint64_t)meas_every - c->sweeps % (uint64_t)meas_every);
            const bool meas_after = meas_every > 0 && (c->sweeps + run) % (uint64_t)meas_every == 0;
            uint32_t *out = overlap && meas_after ? c->spins_alt : c->spins;
            if (overlap && deferred && out == def_buf)               // (a launch in place on the buffer a deferred measurement reads)
                if ((rc = submit_deferred())) return rc;
            if (overlap && c->read_pending[buf_id(out)]) {          // a measurement may still be reading the buffer this launch writes
                if ((rc = check_cuda(c, cudaStreamWaitEvent(c->stream, c->ev_read[buf_id(out)], 0), "wait measurement"))) return rc;
                c->read_pending[buf_id(out)] = false;
            }
            if (c->fail_countdown > 0 && --c->fail_countdown == 0)   // sg_debug_fail_launch: this launch "fails" before it is enqueued
                return fail(c, SG_ECUDA, "sg_run: injected launch failure (sg_debug_fail_launch)");
            const int k = ladder8_supported(c) ? launch_ladder8_pmj(c, c->sweeps, c->exchanges, (int)run, pt_every, out)
                          : gladder_supported(c) ? launch_gladder(c, c->sweeps, (int)run, c->exchanges, pt_every)
                                                 : launch_ladder_pmj(c, c->sweeps, (int)run, c->exchanges, pt_every, out);
            if (k < 0) return check_launch(c, "ladder kernel") ? SG_ECUDA : fail(c, SG_ECUDA, "ladder kernel launch failed");
            if (out != c->spins) std::swap(c->spins, c->spins_alt);
            c->launches += k;
            if (pt_every > 0) c->exchanges += (c->sweeps + run) / (uint64_t)pt_every - c->sweeps / (uint64_t)pt_every;
            c->sweeps += run;
            // the kernel publishes its own energies when an exchange follows its last sweep
            c->um_fresh = pt_every > 0 && c->sweeps % (uint64_t)pt_every == 0;
            left -= (int)run;
            if ((rc = submit_deferred())) return rc;                // the measurement of the state the launch above started from
            if (meas_after) {
                if (overlap) {
                    if ((rc = check_cuda(c, cudaEventRecord(c->ev_state, c->stream), "record state"))) return rc;
                    deferred = true;
                    def_buf = c->spins;
                    def_sweeps = c->sweeps;
                } else if ((rc = do_measure(c, nullptr))) return rc;
            }
        }
        if ((rc = submit_deferred())) return rc;
        if (overlap)                                                  // everything after sg_run is ordered after the measurements
            for (int b = 0; b < 2; ++b)
                if (c->read_pending[b]) {
                    if ((rc = check_cuda(c, cudaStreamWaitEvent(c->stream, c->ev_read[b], 0), "join measurement"))) return rc;
                    c->read_pending[b] = false;
                }
        return SG_OK;
        };
        rc = run_loop();
        if (overlap && rc) {
            // Error exit: the caller's stream must still come after everything the two library streams were given, or a
            // later sg_get_moments / sg_destroy could race a measurement that is still running.  The measurement of the
            // last completed launch is still submitted, so that the counters (sweeps, n_meas) describe the state that
            // is there; then both streams are joined and no read is left marked pending.  The first error is the one
            // reported.
            const std::string first_err = c->err;
            submit_deferred();
            c->stream = user_stream;
            cudaStream_t lib_streams[2] = {c->stream_hi, c->stream2};
            for (cudaStream_t ls : lib_streams)
                if (cudaEventRecord(c->ev_join, ls) == cudaSuccess) cudaStreamWaitEvent(user_stream, c->ev_join, 0);
            c->read_pending[0] = c->read_pending[1] = false;
            c->err = first_err;
            return rc;
        }
        if (overlap) {                                              // ... and the caller's stream continues after both
            c->stream = user_stream;
            if (!rc) rc = check_cuda(c, cudaEventRecord(c->ev_join, c->stream_hi), "record exit");
            if (!rc) rc = check_cuda(c, cudaStreamWaitEvent(user_stream, c->ev_join, 0), "wait exit");
        }
        if (rc) return rc;
        return check_launch(c, "run kernels");
    }
    while (left > 0) {
        // sweeps until the next exchange / measurement is due (or the end)
        uint64_t run = (uint64_t)left;
        if (pt_every > 0) run = std::min<uint64_t>(run, (uint64_t)pt_every - c->sweeps % (uint64_t)pt_every);
        if (meas_every > 0) run = std::min<uint64_t>(run, (uint64_t)meas_every - c->sweeps % (uint64_t)meas_every);
        const bool pt_due = pt_every > 0 && (c->sweeps + run) % (uint64_t)pt_every == 0;
        if (res32_supported(c)) {
            if ((rc = res32_step(c, (int)run, pt_due))) return rc;      // the exchange stays pending for the next launch
        } else {
            if ((rc = do_sweeps(c, (int)run))) return rc;
            if (pt_due)
                if ((rc = do_exchange(c))) return rc;
        }
        left -= (int)run;
        if (meas_every > 0 && c->sweeps % (uint64_t)meas_every == 0)
            if ((rc = do_measure(c, nullptr))) return rc;
    }
    if ((rc = flush_pending(c))) return rc;
    return check_launch(c, "run kernels");
}

int sg_synchronize(sg_ctx *c)
{
    if (!c) return SG_EINVAL;
    return check_cuda(c, cudaStreamSynchronize(c->stream), "sg_synchronize");
}

int sg_destroy(sg_ctx *c)
{
    if (!c) return SG_EINVAL;
    cudaStreamSynchronize(c->stream);
    if (c->stream2) {
        cudaStreamSynchronize(c->stream2);
        cudaEventDestroy(c->ev_state);
        cudaEventDestroy(c->ev_read[0]);
        cudaEventDestroy(c->ev_read[1]);
        cudaStreamDestroy(c->stream2);
        cudaStreamSynchronize(c->stream_hi);
        cudaStreamDestroy(c->stream_hi);
        cudaEventDestroy(c->ev_join);
    }
    if (c->own_ws) cudaFree(c->ws);
    if (c->pq) cudaFree(c->pq);
    if (c->acc_win) cudaFree(c->acc_win);
    delete c;
    return SG_OK;
}

static int spins_range(sg_ctx *c, int s0, int ns, int8_t *out, const int8_t *in)
{
    if (!c) return SG_EINVAL;
    if ((!out && !in) || ns < 1 || s0 < 0 || s0 + ns > c->d.n_samples) return fail(c, SG_EINVAL, "spins range: bad range or NULL buffer");
    const Dims &d = c->d;
    const size_t per = (size_t)d.R * d.NT * d.N;
    const Layout lo = make_layout(d.L, d.n_samples, d.R, d.NT, c->kind);
    {
        const int rc = flush_pending(c);
        if (rc) return rc;
    }
    if (in) {
        c->um_fresh = false;
        if (c->kind == SG_PMJ_TPACK) c->tp_state = 2;
    }
    for (int a = s0; a < s0 + ns; a += lo.chunk_stage) {
        const int n = std::min(lo.chunk_stage, s0 + ns - a);
        int rc;
        if (out) {
            c->launches += is_packed(c) ? launch_unpack_pmj(c, a, n) : launch_unpack_gauss(c, a, n);
            if ((rc = check_launch(c, "unpack kernel"))) return rc;
            if ((rc = check_cuda(c, cudaMemcpyAsync(out + (size_t)(a - s0) * per, c->stage8, per * n, cudaMemcpyDeviceToHost, c->stream), "copy spins"))) return rc;
        } else {
            if ((rc = check_cuda(c, cudaMemcpyAsync(c->stage8, in + (size_t)(a - s0) * per, per * n, cudaMemcpyHostToDevice, c->stream), "copy spins"))) return rc;
            c->launches += is_packed(c) ? launch_pack_pmj(c, a, n) : launch_pack_gauss(c, a, n);
            if ((rc = check_launch(c, "pack kernel"))) return rc;
        }
        if ((rc = check_cuda(c, cudaStreamSynchronize(c->stream), "sync spins"))) return rc;
    }
    return SG_OK;
}

int sg_get_spins_range(sg_ctx *c, int s0, int ns, int8_t *out) { return out ? spins_range(c, s0, ns, out, nullptr) : SG_EINVAL; }
int sg_set_spins_range(sg_ctx *c, int s0, int ns, const int8_t *in) { return in ? spins_range(c, s0, ns, nullptr, in) : SG_EINVAL; }
int sg_get_spins(sg_ctx *c, int8_t *out) { return c ? sg_get_spins_range(c, 0, c->d.n_samples, out) : SG_EINVAL; }
int sg_set_spins(sg_ctx *c, const int8_t *in) { return c ? sg_set_spins_range(c, 0, c->d.n_samples, in) : SG_EINVAL; }

int sg_get_couplings_range(sg_ctx *c, int s0, int ns, float *out)
{
    if (!c) return SG_EINVAL;
    if (!out || ns < 1 || s0 < 0 || s0 + ns > c->d.n_samples) return fail(c, SG_EINVAL, "couplings range: bad range or NULL buffer");
    const Dims &d = c->d;
    const size_t per = (size_t)3 * d.N;
    const Layout lo = make_layout(d.L, d.n_samples, d.R, d.NT, c->kind);
    for (int a = s0; a < s0 + ns; a += lo.chunk_stage) {
        const int n = std::min(lo.chunk_stage, s0 + ns - a);
        float *dev = (float *)c->stage8;
        c->launches += is_packed(c) ? launch_couplings_pmj(c, a, n, dev) : launch_couplings_gauss(c, a, n, dev);
        int rc;
        if ((rc = check_launch(c, "couplings kernel"))) return rc;
        if ((rc = check_cuda(c, cudaMemcpyAsync(out + (size_t)(a - s0) * per, dev, sizeof(float) * per * n, cudaMemcpyDeviceToHost, c->stream), "copy couplings"))) return rc;
        if ((rc = check_cuda(c, cudaStreamSynchronize(c->stream), "sync couplings"))) return rc;
    }
    return SG_OK;
}

int sg_get_couplings(sg_ctx *c, float *out) { return c ? sg_get_couplings_range(c, 0, c->d.n_samples, out) : SG_EINVAL; }

static int copy_energies(sg_ctx *c, int64_t *U, int32_t *M)
{
    int rc;
    const size_t n = (size_t)c->d.n_samples * c->d.R * c->d.NT;
    if (U && (rc = check_cuda(c, cudaMemcpyAsync(U, c->U, sizeof(int64_t) * n, cudaMemcpyDeviceToHost, c->stream), "copy U"))) return rc;
    if (M && (rc = check_cuda(c, cudaMemcpyAsync(M, c->M, sizeof(int32_t) * n, cudaMemcpyDeviceToHost, c->stream), "copy M"))) return rc;
    return check_cuda(c, cudaStreamSynchronize(c->stream), "sync energies");
}

int sg_get_energies(sg_ctx *c, int64_t *U, int32_t *M)
{
    if (!c) return SG_EINVAL;
    int rc;
    if ((rc = flush_pending(c))) return rc;
    c->launches += is_packed(c) ? launch_energy_pmj(c) : launch_energy_gauss(c);     // always a recount
    if ((rc = check_launch(c, "energy kernel"))) return rc;
    c->um_fresh = true;
    return copy_energies(c, U, M);
}

int sg_get_energies_cached(sg_ctx *c, int64_t *U, int32_t *M)
{
    if (!c) return SG_EINVAL;
    if (!c->um_fresh) return fail(c, SG_ESTATE, "sg_get_energies_cached: the kernels' own energies are not up to date with the state");
    int rc;
    if ((rc = flush_pending(c))) return rc;
    return copy_energies(c, U, M);
}

int sg_set_kernel_path(sg_ctx *c, int path)
{
    if (!c) return SG_EINVAL;
    if (path != SG_PATH_AUTO && path != SG_PATH_GENERIC) return fail(c, SG_EINVAL, "sg_set_kernel_path: unknown path");
    const int rc = flush_pending(c);
    if (rc) return rc;
    c->path = path;
    return SG_OK;
}

int sg_get_state_hash(sg_ctx *c, uint64_t *out)
{
    if (!c || !out) return SG_EINVAL;
    int rc;
    if ((rc = flush_pending(c))) return rc;
    c->launches += launch_hash(c, c->hashes);
    if ((rc = check_launch(c, "hash kernel"))) return rc;
    const size_t n = (size_t)c->d.W * c->d.R * c->d.NT;
    if ((rc = check_cuda(c, cudaMemcpyAsync(out, c->hashes, sizeof(uint64_t) * n, cudaMemcpyDeviceToHost, c->stream), "copy hashes"))) return rc;
    return check_cuda(c, cudaStreamSynchronize(c->stream), "sync hashes");
}

// sg_get_state_hash without any allocation: per-system hashes staged in the static device array of sg_noalloc.cu.
// flush_pending only launches kernels into the caller's workspace, so the whole call stays allocation-free.
int sg_get_state_hash_noalloc(sg_ctx *c, uint64_t *out)
{
    if (!c || !out) return SG_EINVAL;
    const long long n_sys = (long long)c->d.W * c->d.R * c->d.NT;
    if (n_sys > (long long)SG_NOALLOC_MAX_SYSTEMS)
        return fail(c, SG_EINVAL, "sg_get_state_hash_noalloc: " + std::to_string(n_sys) + " systems exceed the static scratch of " +
                                      std::to_string((long long)SG_NOALLOC_MAX_SYSTEMS) + " (SG_NOALLOC_MAX_SYSTEMS); use sg_get_state_hash");
    int rc;
    if ((rc = flush_pending(c))) return rc;
    bool too_large = false;
    int launches = 0;
    const cudaError_t e = hash_noalloc(c, out, &too_large, &launches);
    c->launches += (uint64_t)launches;
    if (too_large) return fail(c, SG_EINVAL, "sg_get_state_hash_noalloc: pool exceeds SG_NOALLOC_MAX_SYSTEMS");
    return check_cuda(c, e, "sg_get_state_hash_noalloc");
}

int sg_get_pt_stats(sg_ctx *c, uint64_t *proposed, uint64_t *accepted)
{
    if (!c) return SG_EINVAL;
    const int NT = c->d.NT;
    int rc;
    if ((rc = flush_pending(c))) return rc;
    if (accepted && NT > 1) {
        unsigned long long tmp[MAX_NT];
        if ((rc = check_cuda(c, cudaMemcpyAsync(tmp, c->pt_acc, sizeof(unsigned long long) * MAX_NT, cudaMemcpyDeviceToHost, c->stream), "copy pt counters"))) return rc;
        if ((rc = check_cuda(c, cudaStreamSynchronize(c->stream), "sync pt counters"))) return rc;
        for (int t = 0; t + 1 < NT; ++t) accepted[t] = tmp[t];
    }
    if (proposed) {
        // exchange e proposes the pairs (t, t+1) with t = e mod 2 (R12), once per (sample, replica)
        const uint64_t even = (c->exchanges + 1) / 2, odd = c->exchanges / 2;
        for (int t = 0; t + 1 < NT; ++t) proposed[t] = ((t & 1) ? odd : even) * (uint64_t)c->d.n_samples * (uint64_t)c->d.R;
    }
    return SG_OK;
}

int sg_get_thresholds(sg_ctx *c, uint64_t *out)
{
    if (!c || !out) return SG_EINVAL;
    memcpy(out, c->thr.data(), sizeof(uint64_t) * c->thr.size());
    return SG_OK;
}

int sg_get_moments(sg_ctx *c, double *out, int64_t *n_meas)
{
    if (!c) return SG_EINVAL;
    if (out) {
        const size_t n = (size_t)c->d.n_samples * c->d.NT * SG_NMOM;
        int rc;
        if ((rc = check_cuda(c, cudaMemcpyAsync(out, c->acc, sizeof(double) * n, cudaMemcpyDeviceToHost, c->stream), "copy moments"))) return rc;
        if ((rc = check_cuda(c, cudaStreamSynchronize(c->stream), "sync moments"))) return rc;
    }
    if (n_meas) *n_meas = c->n_meas;
    return SG_OK;
}

int sg_enable_pq(sg_ctx *c, int n_bins)
{
    if (!c) return SG_EINVAL;
    if (n_bins < 1 || n_bins > c->d.N + 1) return fail(c, SG_EINVAL, "sg_enable_pq: need 1 <= n_bins <= N + 1");
    int rc;
    if ((rc = check_cuda(c, cudaStreamSynchronize(c->stream), "sg_enable_pq sync"))) return rc;
    if (c->pq) cudaFree(c->pq);
    c->pq = nullptr;
    c->pq_bins = 0;
    const size_t bytes = sizeof(uint32_t) * (size_t)c->d.n_samples * c->d.NT * n_bins;
    if (cudaMalloc(&c->pq, bytes) != cudaSuccess) { cudaGetLastError(); c->pq = nullptr; return fail(c, SG_ENOMEM, "sg_enable_pq: cudaMalloc failed"); }
    c->pq_bins = n_bins;
    return check_cuda(c, cudaMemsetAsync(c->pq, 0, bytes, c->stream), "zero P(q)");
}

int sg_get_pq(sg_ctx *c, uint32_t *out)
{
    if (!c || !out) return SG_EINVAL;
    if (!c->pq) return fail(c, SG_ESTATE, "sg_get_pq: sg_enable_pq was not called");
    int rc;
    const size_t bytes = sizeof(uint32_t) * (size_t)c->d.n_samples * c->d.NT * c->pq_bins;
    if ((rc = check_cuda(c, cudaMemcpyAsync(out, c->pq, bytes, cudaMemcpyDeviceToHost, c->stream), "copy P(q)"))) return rc;
    return check_cuda(c, cudaStreamSynchronize(c->stream), "sync P(q)");
}

int sg_enable_log_binning(sg_ctx *c, int n_windows)
{
    if (!c) return SG_EINVAL;
    if (n_windows < 1 || n_windows > 40) return fail(c, SG_EINVAL, "sg_enable_log_binning: need 1 <= n_windows <= 40");
    int rc;
    if ((rc = check_cuda(c, cudaStreamSynchronize(c->stream), "sg_enable_log_binning sync"))) return rc;
    if (c->acc_win) cudaFree(c->acc_win);
    c->acc_win = nullptr;
    c->n_windows = 0;
    const size_t bytes = sizeof(double) * (size_t)n_windows * c->d.n_samples * c->d.NT * SG_NMOM;
    if (cudaMalloc(&c->acc_win, bytes) != cudaSuccess) { cudaGetLastError(); c->acc_win = nullptr; return fail(c, SG_ENOMEM, "sg_enable_log_binning: cudaMalloc failed"); }
    c->n_windows = n_windows;
    c->n_meas_win.assign(n_windows, 0);
    return check_cuda(c, cudaMemsetAsync(c->acc_win, 0, bytes, c->stream), "zero windows");
}

int sg_get_window_moments(sg_ctx *c, int k, double *out, int64_t *n_meas)
{
    if (!c) return SG_EINVAL;
    if (!c->acc_win) return fail(c, SG_ESTATE, "sg_get_window_moments: sg_enable_log_binning was not called");
    if (k < 0 || k >= c->n_windows) return fail(c, SG_EINVAL, "sg_get_window_moments: window out of range");
    if (out) {
        const size_t n = (size_t)c->d.n_samples * c->d.NT * SG_NMOM;
        int rc;
        if ((rc = check_cuda(c, cudaMemcpyAsync(out, c->acc_win + (size_t)k * n, sizeof(double) * n, cudaMemcpyDeviceToHost, c->stream), "copy window"))) return rc;
        if ((rc = check_cuda(c, cudaStreamSynchronize(c->stream), "sync window"))) return rc;
    }
    if (n_meas) *n_meas = c->n_meas_win[k];
    return SG_OK;
}

int sg_get_counters(sg_ctx *c, uint64_t *sweeps_done, uint64_t *exchanges_done)
{
    if (!c) return SG_EINVAL;
    if (sweeps_done) *sweeps_done = c->sweeps;
    if (exchanges_done) *exchanges_done = c->exchanges;
    return SG_OK;
}

int sg_set_counters(sg_ctx *c, uint64_t sweeps_done, uint64_t exchanges_done)
{
    if (!c) return SG_EINVAL;
    if (sweeps_done >= (1ull << 31)) return fail(c, SG_EINVAL, "sg_set_counters: the global sweep counter must stay below 2^31");
    const int rc = flush_pending(c);                        // an exchange still pending belongs to the OLD counters
    if (rc) return rc;
    c->sweeps = sweeps_done;
    c->exchanges = exchanges_done;
    c->um_fresh = false;
    return SG_OK;
}

int sg_set_moments(sg_ctx *c, const double *in, int64_t n_meas)
{
    if (!c || !in) return SG_EINVAL;
    if (n_meas < 0) return fail(c, SG_EINVAL, "sg_set_moments: n_meas < 0");
    const size_t n = (size_t)c->d.n_samples * c->d.NT * SG_NMOM;
    int rc;
    if ((rc = check_cuda(c, cudaMemcpyAsync(c->acc, in, sizeof(double) * n, cudaMemcpyHostToDevice, c->stream), "copy moments"))) return rc;
    if ((rc = check_cuda(c, cudaStreamSynchronize(c->stream), "sync moments"))) return rc;
    c->n_meas = n_meas;
    return SG_OK;
}

int sg_get_launch_count(sg_ctx *c, uint64_t *launches)
{
    if (!c || !launches) return SG_EINVAL;
    *launches = c->launches;
    return SG_OK;
}

int sg_get_accept_variant(sg_ctx *c, int *variant)
{
    if (!c || !variant) return SG_EINVAL;
    if (c->kind == SG_GAUSS) return fail(c, SG_EUNSUPPORTED, "sg_get_accept_variant: +-J kinds only");
    *variant = c->d.bs_accept ? SG_ACCEPT_BINARY_SEARCH : c->d.fast_accept ? SG_ACCEPT_CARRY_CHAIN : SG_ACCEPT_GENERAL;
    return SG_OK;
}

int sg_debug_fail_launch(sg_ctx *c, int countdown)
{
    if (!c) return SG_EINVAL;
    if (countdown < 0) return fail(c, SG_EINVAL, "sg_debug_fail_launch: countdown < 0");
    c->fail_countdown = countdown;
    return SG_OK;
}

const char *sg_last_error(sg_ctx *c) { return c ? c->err.c_str() : g_create_err.c_str(); }

}  // extern "C"
