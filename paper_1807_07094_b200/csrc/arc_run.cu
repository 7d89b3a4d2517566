// arc_run.cu -- the compute entry points of include/arc.h: arc_trace, arc_update_chemistry, and the
// read-back calls.  Launch order of one trace: scheduler reset -> a1+a2 opacity/zero ->
// a3-a9 persistent tracer -> a10 finalize.  All on the context's stream; CUDA events bracket each kernel so
// that callers (bench.py) can read per-kernel device times measured on the launching stream.
#include "arc_internal.cuh"
#include <cmath>
#include <cstring>
#include <vector>

#define CK(call)                                                                                              \
    do {                                                                                                      \
        cudaError_t e_ = (call);                                                                              \
        if (e_ != cudaSuccess) {                                                                              \
            c->err = std::string(#call) + ": " + cudaGetErrorString(e_);                                      \
            return e_ == cudaErrorMemoryAllocation ? ARC_ENOMEM : ARC_ECUDA;                                  \
        }                                                                                                     \
    } while (0)

static int fail(arc_ctx *c, int code, const std::string &msg) { c->err = msg; return code; }

static size_t famrec_bytes(int nb) { return (size_t)(16 + 16 * nb); }      // sizeof(FamRec<nb>)

// check the device-side error word after the stream has been synchronised; an error is reported once and cleared (the
// word is sticky on the device: until then every consumer kernel skips its work, arc_trace.cu / arc_fields.cu / arc_chem.cu)
int arc_check_device(arc_ctx *c)
{
    c->unchecked = false;
    SchedState h;
    CK(cudaMemcpy(&h, c->d_sched, sizeof(h), cudaMemcpyDeviceToHost));
    if (h.error == ARC_DEV_OK && h.in_flight == 0) return ARC_OK;
    c->have_rates = false; c->have_accum = false;
    c->queue_dirty = true;                        // families may be left in the donation queue: full reset before the next trace
    CK(cudaMemset(&c->d_sched->error, 0, sizeof(int)));
    switch (h.error) {
        case ARC_DEV_STACK_OVERFLOW: return fail(c, ARC_EOVERFLOW, "arc_trace: a warp's work stack overflowed; rates are invalid");
        case ARC_DEV_LOG_OVERFLOW: return fail(c, ARC_EOVERFLOW, "arc_trace_debug: ray log too small");
        case ARC_DEV_WATCHDOG: return fail(c, ARC_ECUDA, "arc_trace: scheduler watchdog fired (no progress for 20 s); rates are invalid");
        case ARC_DEV_RAY_RUNAWAY: return fail(c, ARC_ECUDA, "arc_trace: a ray exceeded 3N+8 segments; rates are invalid");
        case ARC_DEV_CHECK_FAILED: return fail(c, ARC_ECUDA, "arc_trace: a bounds check of the checked build failed; rates are invalid");
        default: return fail(c, ARC_ECUDA, "arc_trace: kernel ended with work still in flight; rates are invalid");
    }
}

// host side of a trace: state checks, (re)allocation of the work stacks and the queue, the kernel's arguments, and - with
// an optically thin region - the per-source start radii.  Nothing is enqueued except those small copies.
static int prepare_trace(arc_ctx *c, arc_raylog *log, unsigned long long *d_key, unsigned int *d_seq, int *d_cell, TraceArgs &a, double &thin_maxR)
{
    if (!c->have_fields) return fail(c, ARC_ESTATE, "arc_trace: no fields set (arc_set_fields)");
    if (!c->have_spec) return fail(c, ARC_ESTATE, "arc_trace: no spectrum set (arc_set_spectrum)");
    if (!c->have_src) return fail(c, ARC_ESTATE, "arc_trace: no sources set (arc_set_sources)");
    if (c->d_blocked && c->mask_level != c->p.l0) return fail(c, ARC_ESTATE, "arc_trace: the emission mask was set for another l0 (arc_set_emission_mask)");
    const int nb = c->spec.nb;
    // persistent grid: what is co-resident (SM count x blocks per SM), or the caller's override
    const bool thin = c->p.thin_tau > 0.0;
    if (thin && log) return fail(c, ARC_EINVAL, "arc_trace_debug: the per-ray log is not built for thin_tau > 0");
    const int flags = (log ? 3 : (c->p.digest ? 2 : 0)) | (c->p.geom_corr ? 4 : 0) | (thin ? 8 : 0);     // FLAG_LOG 1, FLAG_DIGEST 2, FLAG_GEOM 4, FLAG_THIN 8
    const int resident = arc_trace_occupancy_grid(c, nb, flags);
    int grid = c->p.trace_blocks > 0 ? c->p.trace_blocks : resident;
    if (grid > resident) grid = resident;         // blocks wait on one another: never oversubscribe
    if (grid < 1) grid = 1;
    c->trace_grid = grid;
    const size_t rec = famrec_bytes(nb);
    const size_t need_stacks = (size_t)grid * ARC_WARPS_PER_BLOCK * ARC_STACK_CAP * rec;
    const size_t need_queue = (size_t)ARC_QUEUE_CAP * rec;
    if (need_stacks > c->stacks_bytes) {
        CK(cudaStreamSynchronize(c->stream));
        cudaFree(c->d_stacks); c->d_stacks = nullptr; c->stacks_bytes = 0;
        CK(cudaMalloc(&c->d_stacks, need_stacks));
        c->stacks_bytes = need_stacks; ++c->epoch;
    }
    if (need_queue > c->queue_bytes) {
        CK(cudaStreamSynchronize(c->stream));
        cudaFree(c->d_queue); c->d_queue = nullptr; c->queue_bytes = 0;
        CK(cudaMalloc(&c->d_queue, need_queue));
        c->queue_bytes = need_queue; ++c->epoch;
    }
    if (!c->d_qseq) { CK(cudaMalloc(&c->d_qseq, sizeof(unsigned long long) * ARC_QUEUE_CAP)); c->queue_dirty = true; }

    std::memset(&a, 0, sizeof(a));
    a.N = c->N; a.NN = c->N * c->N; a.max_seg = 3u * (unsigned)c->N + 8u; a.nb = nb; a.nbp = arc_nbp(nb); a.l0 = c->p.l0; a.Lmax = c->p.Lmax; a.nsrc = c->nsrc;
    a.dx = c->dx;
    a.csplit = std::sqrt(3.0 / (3.14159265358979323846 * c->p.Phi));      // O2: r_split(l) = csplit 2^l cells
    a.tau_term = c->p.tau_term;
    a.cpix = std::sqrt(3.14159265358979323846 / 3.0);                     // sqrt(Omega_l) = cpix 2^-l (G26)
    a.geom = c->p.geom_corr;
    a.kappa = c->d_kappa; a.A = c->d_A; a.src_g = c->d_src_g; a.src_S = c->d_src_S; a.blocked = c->d_blocked;
    a.stacks = c->d_stacks; a.queue = c->d_queue; a.qseq = c->d_qseq; a.sched = c->d_sched; a.stats = c->d_stats;
    a.fam_per_src = 3u << (2 * c->p.l0);
    a.seed_total = (unsigned long long)c->nsrc * a.fam_per_src;
    thin_maxR = 0.0;
    if (thin && c->nsrc > 0) {
        // optically thin inner region: per source, the radius the last trace found, the level rays have
        // there (r_split(l-1) <= R < r_split(l)), its root families, and the rate the open root rays carry together
        const int ns = c->nsrc;
        if (c->thin_cap < ns) {
            CK(cudaStreamSynchronize(c->stream));
            cudaFree(c->d_Rstart); cudaFree(c->d_Rnext); cudaFree(c->d_seed_prefix); cudaFree(c->d_src_level); cudaFree(c->d_Sopen);
            c->d_Rstart = nullptr; c->d_Rnext = nullptr; c->d_seed_prefix = nullptr; c->d_src_level = nullptr; c->d_Sopen = nullptr; c->thin_cap = 0;
            CK(cudaMalloc(&c->d_Rstart, sizeof(double) * ns));
            CK(cudaMalloc(&c->d_Rnext, sizeof(unsigned long long) * ns));
            CK(cudaMalloc(&c->d_seed_prefix, sizeof(unsigned long long) * (ns + 1)));
            CK(cudaMalloc(&c->d_src_level, sizeof(int) * ns));
            CK(cudaMalloc(&c->d_Sopen, sizeof(double) * ns * ARC_MAX_BINS));
            c->thin_cap = ns;
        }
        std::vector<unsigned long long> prefix((size_t)ns + 1), inf((size_t)ns, 0x7ff0000000000000ull);
        std::vector<int> lev((size_t)ns);
        std::vector<double> Sopen((size_t)ns * nb);
        const double npix0 = (double)(12ull << (2 * c->p.l0));
        prefix[0] = 0;
        for (int s = 0; s < ns; ++s) {
            const double R = c->h_R[(size_t)s];
            int l = c->p.l0;
            if (R > 0.0) while (l < c->p.Lmax && std::ldexp(a.csplit, l) <= R) ++l;
            lev[(size_t)s] = l;
            prefix[(size_t)s + 1] = prefix[(size_t)s] + (3ull << (2 * l));
            if (R > thin_maxR) thin_maxR = R;
            const double nopen = c->h_nopen[(size_t)s] < 0.0 ? npix0 : c->h_nopen[(size_t)s];
            for (int v = 0; v < nb; ++v) Sopen[(size_t)s * nb + v] = c->h_src_S[(size_t)s * nb + v] / npix0 * nopen;
        }
        CK(cudaMemcpyAsync(c->d_Rstart, c->h_R.data(), sizeof(double) * ns, cudaMemcpyHostToDevice, c->stream));
        CK(cudaMemcpyAsync(c->d_Rnext, inf.data(), sizeof(unsigned long long) * ns, cudaMemcpyHostToDevice, c->stream));
        CK(cudaMemcpyAsync(c->d_seed_prefix, prefix.data(), sizeof(unsigned long long) * (ns + 1), cudaMemcpyHostToDevice, c->stream));
        CK(cudaMemcpyAsync(c->d_src_level, lev.data(), sizeof(int) * ns, cudaMemcpyHostToDevice, c->stream));
        CK(cudaMemcpyAsync(c->d_Sopen, Sopen.data(), sizeof(double) * ns * nb, cudaMemcpyHostToDevice, c->stream));
        CK(cudaStreamSynchronize(c->stream));                        // (the host vectors go out of scope)
        a.thin_tau = c->p.thin_tau; a.Rstart = c->d_Rstart; a.Rnext = c->d_Rnext; a.seed_prefix = c->d_seed_prefix; a.src_level = c->d_src_level;
        a.seed_total = prefix[(size_t)ns];
    }
    {   // few sources: spread the root families over the warps instead of 8 per warp
        const unsigned long long per_warp = a.seed_total / ((unsigned long long)grid * ARC_WARPS_PER_BLOCK);
        a.seed_chunk = per_warp >= ARC_BATCH_FAM ? ARC_BATCH_FAM : (per_warp < 1 ? 1 : (int)per_warp);
    }
    a.flags = flags;
    a.log_key = d_key; a.log_seq = d_seq; a.log_cell = d_cell; a.log_cap = log ? (unsigned long long)log->cap : 0ull;
    return ARC_OK;
}

// the kernels of one trace, in stream order: [queue reset if needed] -> a1 + a2 + per-trace reset -> [thin region] ->
// a3-a9 persistent tracer -> a10 finalize.  `events`: bracket them with the context's CUDA events (not inside a graph capture).
static int enqueue_trace(arc_ctx *c, const TraceArgs &a, bool log, bool finalize, double thin_maxR, bool events)
{
    if (c->queue_dirty) { CK(arc_launch_queue_reset(c)); c->queue_dirty = false; }
    if (events) CK(cudaEventRecord(c->ev[0], c->stream));
    CK(arc_launch_opacity(c, a.seed_total));
    if (thin_maxR > 0.0) CK(arc_launch_thin_region(c, thin_maxR));          // (iii): after the accumulators are zeroed
    if (events) CK(cudaEventRecord(c->ev[1], c->stream));
    CK(arc_launch_trace(c, a, log, nullptr));
    if (events) CK(cudaEventRecord(c->ev[2], c->stream));
    if (finalize) CK(arc_launch_finalize(c));          // arc_trace_partial leaves a10 to arc_finalize
    if (events) CK(cudaEventRecord(c->ev[3], c->stream));
    return ARC_OK;
}

static int run_trace(arc_ctx *c, arc_raylog *log, unsigned long long *d_key, unsigned int *d_seq, int *d_cell, bool finalize = true)
{
    TraceArgs a; double thin_maxR = 0.0;
    { const int rc = prepare_trace(c, log, d_key, d_seq, d_cell, a, thin_maxR); if (rc != ARC_OK) return rc; }
    const bool thin = c->p.thin_tau > 0.0;
    { const int rc = enqueue_trace(c, a, log != nullptr, finalize, thin ? thin_maxR : 0.0, true); if (rc != ARC_OK) return rc; }
    c->traced_once = true; c->steps_timed = false;
    c->have_rates = finalize;
    c->have_accum = !finalize;
    c->finalize_split = false;
    if (thin && c->nsrc > 0) {                 // (ii): the radii this trace found are the next trace's
        std::vector<unsigned long long> bits((size_t)c->nsrc);
        CK(cudaMemcpyAsync(bits.data(), c->d_Rnext, sizeof(unsigned long long) * c->nsrc, cudaMemcpyDeviceToHost, c->stream));
        CK(cudaStreamSynchronize(c->stream));
        const int de = arc_check_device(c);
        if (de != ARC_OK) return de;
        for (int s = 0; s < c->nsrc; ++s) {
            double R = 0.0;
            if (bits[(size_t)s] < 0x7ff0000000000000ull) std::memcpy(&R, &bits[(size_t)s], sizeof(R));
            c->h_R[(size_t)s] = R;
        }
        return ARC_OK;
    }
    if (!c->p.async || log) {
        CK(cudaStreamSynchronize(c->stream));
        return arc_check_device(c);
    }
    c->unchecked = true;              // async: whoever synchronises next looks at the device error word
    return ARC_OK;
}

// for the calls that have just synchronised the stream
static int check_pending(arc_ctx *c) { return c->unchecked ? arc_check_device(c) : ARC_OK; }

static void fill_rates(arc_ctx *c, arc_rates *out)
{
    const double *r = c->d_rates;
    const int64_t n = c->ncell;
    out->Gamma_HI = r; out->Gamma_HeI = r + n; out->Gamma_HeII = r + 2 * n;
    out->heat_HI = r + 3 * n; out->heat_HeI = r + 4 * n; out->heat_HeII = r + 5 * n;
    out->heat_total = r + 6 * n;
}

extern "C" {

int arc_trace(arc_ctx *c, int step, arc_rates *out)
{
    (void)step;
    if (!c) return ARC_EINVAL;
    const int rc = run_trace(c, nullptr, nullptr, nullptr, nullptr);
    if (rc == ARC_OK && out) fill_rates(c, out);
    return rc;
}

int arc_trace_partial(arc_ctx *c, int step)
{
    (void)step;
    if (!c) return ARC_EINVAL;
    return run_trace(c, nullptr, nullptr, nullptr, nullptr, false);
}

int arc_accum_device(arc_ctx *c, double **A, int64_t *n_doubles)
{
    if (!c || !A || !n_doubles) return ARC_EINVAL;
    if (!c->have_spec) return fail(c, ARC_ESTATE, "arc_accum_device: no spectrum set (the record length is the bin count)");
    *A = c->d_A;
    *n_doubles = (int64_t)c->ncell * arc_nbp(c->spec.nb);
    return ARC_OK;
}

int arc_finalize(arc_ctx *c, arc_rates *out)
{
    if (!c) return ARC_EINVAL;
    if (!c->have_accum) return fail(c, ARC_ESTATE, "arc_finalize: no partial trace to finalise (call arc_trace_partial; setting fields, sources, spectrum or parameters discards it)");
    CK(cudaEventRecord(c->ev[4], c->stream));
    CK(arc_launch_finalize(c));
    CK(cudaEventRecord(c->ev[7], c->stream));
    c->have_accum = false;
    c->have_rates = true;
    c->finalize_split = true;
    if (!c->p.async) { CK(cudaStreamSynchronize(c->stream)); const int de = check_pending(c); if (de != ARC_OK) return de; }
    if (out) fill_rates(c, out);
    return ARC_OK;
}

int arc_trace_debug(arc_ctx *c, int step, arc_raylog *log)
{
    (void)step;
    if (!c || !log) return ARC_EINVAL;
    if (log->cap < 1 || !log->key || !log->seq || !log->cell) return fail(c, ARC_EINVAL, "arc_trace_debug: log buffers missing");
    unsigned long long *d_key = nullptr; unsigned int *d_seq = nullptr; int *d_cell = nullptr;
    log->n = 0;
    cudaError_t e = cudaMalloc(&d_key, sizeof(unsigned long long) * log->cap);
    if (e == cudaSuccess) e = cudaMalloc(&d_seq, sizeof(unsigned int) * log->cap);
    if (e == cudaSuccess) e = cudaMalloc(&d_cell, sizeof(int) * log->cap);
    int rc = ARC_OK;
    if (e != cudaSuccess) { cudaGetLastError(); rc = fail(c, ARC_ENOMEM, "arc_trace_debug: cannot allocate the device log"); }
    if (rc == ARC_OK) rc = run_trace(c, log, d_key, d_seq, d_cell);
    if (rc == ARC_OK) {
        SchedState h;
        e = cudaMemcpy(&h, c->d_sched, sizeof(h), cudaMemcpyDeviceToHost);
        if (e == cudaSuccess) {
            log->n = (int64_t)h.log_n;
            if (h.log_n > (unsigned long long)log->cap) { c->have_rates = false; rc = fail(c, ARC_EOVERFLOW, "arc_trace_debug: ray log too small (log->n holds the size needed)"); }
        }
        if (e == cudaSuccess && rc == ARC_OK) e = cudaMemcpy(log->key, d_key, sizeof(unsigned long long) * log->n, cudaMemcpyDeviceToHost);
        if (e == cudaSuccess && rc == ARC_OK) e = cudaMemcpy(log->seq, d_seq, sizeof(unsigned int) * log->n, cudaMemcpyDeviceToHost);
        if (e == cudaSuccess && rc == ARC_OK) e = cudaMemcpy(log->cell, d_cell, sizeof(int) * log->n, cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) rc = fail(c, ARC_ECUDA, std::string("arc_trace_debug: ") + cudaGetErrorString(e));
    }
    cudaFree(d_key); cudaFree(d_seq); cudaFree(d_cell);
    return rc;
}

int arc_get_rates(arc_ctx *c, double *Gamma_HI, double *Gamma_HeI, double *Gamma_HeII, double *heat_HI, double *heat_HeI,
                  double *heat_HeII, double *heat_total, int where)
{
    if (!c) return ARC_EINVAL;
    if (where != ARC_HOST && where != ARC_DEVICE) return fail(c, ARC_EINVAL, "arc_get_rates: bad `where`");
    if (!c->have_rates) return fail(c, ARC_ESTATE, "arc_get_rates: no valid rates (call arc_trace)");
    double *dst[7] = {Gamma_HI, Gamma_HeI, Gamma_HeII, heat_HI, heat_HeI, heat_HeII, heat_total};
    const cudaMemcpyKind kind = (where == ARC_HOST) ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice;
    for (int i = 0; i < 7; ++i)
        if (dst[i]) CK(cudaMemcpyAsync(dst[i], c->d_rates + (size_t)i * c->ncell, (size_t)c->ncell * sizeof(double), kind, c->stream));
    if (where == ARC_HOST) { CK(cudaStreamSynchronize(c->stream)); return check_pending(c); }
    return ARC_OK;
}

int arc_get_accum(arc_ctx *c, double *A, int where)
{
    if (!c || !A) return ARC_EINVAL;
    if (where != ARC_HOST && where != ARC_DEVICE) return fail(c, ARC_EINVAL, "arc_get_accum: bad `where`");
    if (!c->have_rates && !c->have_accum) return fail(c, ARC_ESTATE, "arc_get_accum: no valid trace (call arc_trace)");
    const cudaMemcpyKind kind = (where == ARC_HOST) ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice;
    const int nb = c->spec.nb, nbp = arc_nbp(nb);        // device rows are padded to nbp doubles; the caller gets [cell][nb]
    if (nbp == nb) CK(cudaMemcpyAsync(A, c->d_A, (size_t)c->ncell * nb * sizeof(double), kind, c->stream));
    else CK(cudaMemcpy2DAsync(A, nb * sizeof(double), c->d_A, nbp * sizeof(double), nb * sizeof(double), (size_t)c->ncell, kind, c->stream));
    if (where == ARC_HOST) { CK(cudaStreamSynchronize(c->stream)); return check_pending(c); }
    return ARC_OK;
}

static int enqueue_chemistry(arc_ctx *c, double dt_s, bool events)
{
    if (events) CK(cudaEventRecord(c->ev[5], c->stream));
    CK(cudaMemsetAsync(&c->d_stats->subcycles, 0, 2 * sizeof(unsigned long long) + 2 * sizeof(unsigned int), c->stream));
    CK(arc_launch_chemistry(c, dt_s));
    if (events) CK(cudaEventRecord(c->ev[6], c->stream));
    return ARC_OK;
}

int arc_run_steps(arc_ctx *c, int n_steps, double dt_s)
{
    if (!c) return ARC_EINVAL;
    if (n_steps < 1) return fail(c, ARC_EINVAL, "arc_run_steps: n_steps must be >= 1");
    if (!(dt_s >= 0.0) || !std::isfinite(dt_s)) return fail(c, ARC_EINVAL, "arc_run_steps: dt must be finite and >= 0");
    if (c->p.thin_tau > 0.0) return fail(c, ARC_EINVAL, "arc_run_steps: not built for thin_tau > 0 (every trace hands its radii to the host)");
    TraceArgs a; double thin_maxR = 0.0;
    { const int rc = prepare_trace(c, nullptr, nullptr, nullptr, nullptr, a, thin_maxR); if (rc != ARC_OK) return rc; }
    if (!c->ev_steps[0]) { CK(cudaEventCreate(&c->ev_steps[0])); CK(cudaEventCreate(&c->ev_steps[1])); }
    if (c->queue_dirty) { CK(arc_launch_queue_reset(c)); c->queue_dirty = false; }
    // one step = the kernels of arc_trace + arc_update_chemistry; captured once into a CUDA graph (a user stream is needed:
    // the legacy default stream cannot be captured - the steps are then enqueued one by one, still without a host round trip)
    const bool use_graph = c->stream != nullptr;
    if (use_graph && (!c->step_exec || c->step_epoch != c->epoch || c->step_dt != dt_s)) {
        if (c->step_exec) { cudaGraphExecDestroy(c->step_exec); c->step_exec = nullptr; }
        cudaGraph_t g = nullptr;
        const unsigned long long l0 = c->launches;
        CK(cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal));
        int rc = enqueue_trace(c, a, false, true, 0.0, false);
        if (rc == ARC_OK) rc = enqueue_chemistry(c, dt_s, false);
        const cudaError_t e = cudaStreamEndCapture(c->stream, &g);
        if (rc != ARC_OK || e != cudaSuccess) { if (g) cudaGraphDestroy(g); cudaGetLastError(); return rc != ARC_OK ? rc : fail(c, ARC_ECUDA, std::string("arc_run_steps: graph capture: ") + cudaGetErrorString(e)); }
        c->step_launches = c->launches - l0; c->launches = l0;        // (captured, not launched)
        const cudaError_t e2 = cudaGraphInstantiate(&c->step_exec, g, 0);
        cudaGraphDestroy(g);
        if (e2 != cudaSuccess) { c->step_exec = nullptr; return fail(c, ARC_ECUDA, std::string("arc_run_steps: cudaGraphInstantiate: ") + cudaGetErrorString(e2)); }
        c->step_epoch = c->epoch; c->step_dt = dt_s;
    }
    CK(cudaEventRecord(c->ev_steps[0], c->stream));
    for (int i = 0; i < n_steps; ++i) {
        if (use_graph) { CK(cudaGraphLaunch(c->step_exec, c->stream)); c->launches += c->step_launches; }
        else {
            int rc = enqueue_trace(c, a, false, true, 0.0, false);
            if (rc == ARC_OK) rc = enqueue_chemistry(c, dt_s, false);
            if (rc != ARC_OK) return rc;
        }
    }
    CK(cudaEventRecord(c->ev_steps[1], c->stream));
    c->traced_once = true; c->chem_once = true; c->steps_timed = true;
    c->have_rates = true; c->have_accum = false; c->finalize_split = false;
    if (!c->p.async) { CK(cudaStreamSynchronize(c->stream)); return arc_check_device(c); }
    c->unchecked = true;
    return ARC_OK;
}

int arc_update_chemistry(arc_ctx *c, double dt_s)
{
    if (!c) return ARC_EINVAL;
    if (!(dt_s >= 0.0) || !std::isfinite(dt_s)) return fail(c, ARC_EINVAL, "arc_update_chemistry: dt must be finite and >= 0");
    if (!c->have_rates) return fail(c, ARC_ESTATE, "arc_update_chemistry: no valid rates (call arc_trace after setting fields)");
    { const int rc = enqueue_chemistry(c, dt_s, true); if (rc != ARC_OK) return rc; }
    c->chem_once = true;
    // the rates stay valid as numbers, but they belong to the fields before this update
    if (!c->p.async) { CK(cudaStreamSynchronize(c->stream)); return check_pending(c); }
    return ARC_OK;
}

int arc_suggest_dt(arc_ctx *c, int scheme, double eps, double *dt_s, int64_t *cells_used)
{
    if (!c) return ARC_EINVAL;
    if (!dt_s) return fail(c, ARC_EINVAL, "arc_suggest_dt: dt_s is NULL");
    if (scheme != ARC_DT_NEUTRAL && scheme != ARC_DT_INTENSITY) return fail(c, ARC_EINVAL, "arc_suggest_dt: scheme must be ARC_DT_NEUTRAL or ARC_DT_INTENSITY");
    if (!(eps > 0.0) || !std::isfinite(eps)) return fail(c, ARC_EINVAL, "arc_suggest_dt: eps must be finite and > 0");
    if (!c->have_rates) return fail(c, ARC_ESTATE, "arc_suggest_dt: no valid rates (call arc_trace after setting fields)");
    if (!c->d_dt) CK(cudaMalloc(&c->d_dt, 2 * sizeof(unsigned long long)));
    CK(cudaMemsetAsync(c->d_dt, 0xFF, sizeof(unsigned long long), c->stream));        // above the bits of +inf
    CK(cudaMemsetAsync(c->d_dt + 1, 0, sizeof(unsigned long long), c->stream));
    CK(arc_launch_suggest_dt(c, scheme, eps));
    unsigned long long h[2];
    CK(cudaMemcpyAsync(h, c->d_dt, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    { const int de = check_pending(c); if (de != ARC_OK) return de; }
    double dt = INFINITY;
    if (h[0] < 0x7ff0000000000000ull) std::memcpy(&dt, &h[0], sizeof(dt));
    *dt_s = dt;
    if (cells_used) *cells_used = (int64_t)h[1];
    return ARC_OK;
}

int arc_synchronize(arc_ctx *c)
{
    if (!c) return ARC_EINVAL;
    CK(cudaStreamSynchronize(c->stream));
    if (c->traced_once) return arc_check_device(c);
    return ARC_OK;
}

int arc_get_stats(arc_ctx *c, arc_stats *s)
{
    if (!c || !s) return ARC_EINVAL;
    std::memset(s, 0, sizeof(*s));
    CK(cudaStreamSynchronize(c->stream));
    DevStats d; SchedState h; double ab[ARC_MAX_BINS];
    CK(cudaMemcpy(&d, c->d_stats, sizeof(d), cudaMemcpyDeviceToHost));
    CK(cudaMemcpy(&h, c->d_sched, sizeof(h), cudaMemcpyDeviceToHost));
    CK(cudaMemcpy(ab, c->d_absorbed, sizeof(ab), cudaMemcpyDeviceToHost));
    s->deposit_records = d.deposit_records; s->segments = d.segments; s->rays = d.rays; s->digest = d.digest; s->queue_high_water = h.q_high;
    for (int l = 0; l < ARC_MAX_LEVEL; ++l) { s->splits[l] = d.splits[l]; s->rays_level[l] = d.rays_level[l]; }
    for (int i = 0; i < 3; ++i) s->ends[i] = d.ends[i];
    for (int v = 0; v < ARC_MAX_BINS; ++v) { s->emitted[v] = c->have_src ? c->emitted[v] : 0.0; s->absorbed[v] = ab[v]; s->escaped[v] = d.escaped[v]; }
    s->subcycles = d.subcycles; s->max_subcycles_cell = d.max_sub;
    s->trace_grid = c->trace_grid;
    s->segments_total = d.segments_total; s->subcycles_total = d.subcycles_total;
    if (c->steps_timed) cudaEventElapsedTime(&s->steps_ms, c->ev_steps[0], c->ev_steps[1]);     // (per-kernel times: not inside a graph)
    else if (c->traced_once) {
        cudaEventElapsedTime(&s->trace_ms, c->ev[0], c->ev[3]);
        cudaEventElapsedTime(&s->opacity_ms, c->ev[0], c->ev[1]);
        cudaEventElapsedTime(&s->trace_kernel_ms, c->ev[1], c->ev[2]);
        cudaEventElapsedTime(&s->finalize_ms, c->ev[2], c->ev[3]);
        if (c->finalize_split) {                  // arc_trace_partial + arc_finalize: the finalise pass was timed on its own
            cudaEventElapsedTime(&s->finalize_ms, c->ev[4], c->ev[7]);
            s->trace_ms += s->finalize_ms;
        }
    }
    if (c->chem_once && !c->steps_timed) cudaEventElapsedTime(&s->chem_ms, c->ev[5], c->ev[6]);
    s->kernel_launches = c->launches;
    cudaGetLastError();
    return check_pending(c);                    // (the statistics are filled in either way)
}

int arc_pix2vec(const int32_t *level, const uint32_t *pix, int n, double *out)
{
    if (n < 0 || (n > 0 && (!level || !pix || !out))) return ARC_EINVAL;
    if (n == 0) return ARC_OK;
    for (int i = 0; i < n; ++i)
        if (level[i] < 0 || level[i] > 14 || (unsigned long long)pix[i] >= (12ull << (2 * level[i]))) return ARC_EINVAL;
    int32_t *d_l = nullptr; uint32_t *d_p = nullptr; double *d_o = nullptr;
    cudaError_t e = cudaMalloc(&d_l, sizeof(int32_t) * n);
    if (e == cudaSuccess) e = cudaMalloc(&d_p, sizeof(uint32_t) * n);
    if (e == cudaSuccess) e = cudaMalloc(&d_o, sizeof(double) * 3 * n);
    if (e == cudaSuccess) e = cudaMemcpy(d_l, level, sizeof(int32_t) * n, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(d_p, pix, sizeof(uint32_t) * n, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = arc_launch_pix2vec(d_l, d_p, n, d_o, 0);
    if (e == cudaSuccess) e = cudaMemcpy(out, d_o, sizeof(double) * 3 * n, cudaMemcpyDeviceToHost);
    cudaFree(d_l); cudaFree(d_p); cudaFree(d_o);
    if (e != cudaSuccess) { cudaGetLastError(); return ARC_ECUDA; }
    return ARC_OK;
}

}  // extern "C"
