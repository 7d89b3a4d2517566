// arc_trace.cu -- host side of the persistent tracer: deposit-mode choice, dispatch to the instantiation units
// (arc_trace_inst_*.cu), scheduler reset and the exposed pix2vec kernel.  The kernel itself is arc_trace_kernel.cuh.
#include "arc_internal.cuh"
#include "arc_healpix.cuh"

#define DECL_INST(tag)                                                                                        \
    cudaError_t arc_trace_launch_##tag(const TraceArgs &a, bool log, int dep, int grid, cudaStream_t s);      \
    int arc_trace_occ_##tag(int nb, int dep, int flags);
DECL_INST(f32_lo) DECL_INST(f32_hi) DECL_INST(f64_lo) DECL_INST(f64_hi)

namespace {

// scheduler reset before each trace: all root families are "in flight", queue empty, slot i expects ticket i
__global__ void arc_sched_reset_kernel(SchedState *sc, DevStats *st, unsigned long long *qseq, unsigned long long seed_total)
{
    const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < ARC_QUEUE_CAP) qseq[i] = i;
    if (i == 0) {
        sc->in_flight = (long long)seed_total; sc->seed_next = 0; sc->q_head = 0; sc->q_tail = 0;
        sc->hungry = 0; sc->error = ARC_DEV_OK; sc->q_high = 0; sc->log_n = 0; sc->q_count = 0;
        st->segments = 0; st->rays = 0; st->digest = 0; st->deposit_records = 0;
        for (int l = 0; l < ARC_MAX_LEVEL; ++l) { st->splits[l] = 0; st->rays_level[l] = 0; }
        for (int e = 0; e < 3; ++e) st->ends[e] = 0;
        for (int v = 0; v < ARC_MAX_BINS; ++v) st->escaped[v] = 0.0;
    }
}

__global__ void arc_pix2vec_kernel(const int32_t *level, const uint32_t *pix, int n, double *out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double x, y, z;
    arc_pix2vec_dev(level[i], pix[i], x, y, z);
    out[3 * i] = x; out[3 * i + 1] = y; out[3 * i + 2] = z;
}


}  // namespace

// ARC_DEPOSIT_* -> the kernel's DEP_* (1 RED, 2 AGG, 3 T).  AUTO: see DESIGN.md 6.2 for the measurements behind it.
int arc_trace_deposit_mode(const arc_ctx *c, int nb)
{
    if (c->p.deposit != ARC_DEPOSIT_AUTO) return c->p.deposit;
    return nb >= 3 ? 3 : 2;
}

int arc_trace_occupancy_grid(arc_ctx *c, int nb, int flags)
{
    const int dep = arc_trace_deposit_mode(c, nb);
    int per_sm;                          // co-resident blocks of exactly the variant that will be launched
    if (c->dtype == ARC_F32) per_sm = nb <= 4 ? arc_trace_occ_f32_lo(nb, dep, flags) : arc_trace_occ_f32_hi(nb, dep, flags);
    else per_sm = nb <= 4 ? arc_trace_occ_f64_lo(nb, dep, flags) : arc_trace_occ_f64_hi(nb, dep, flags);
    return c->n_sm * per_sm;
}

cudaError_t arc_launch_trace(arc_ctx *c, const TraceArgs &a, bool log, int *grid_out)
{
    const int grid = c->trace_grid;
    if (grid_out) *grid_out = grid;
    const int dep = arc_trace_deposit_mode(c, a.nb);
    if (c->dtype == ARC_F32)
        return a.nb <= 4 ? arc_trace_launch_f32_lo(a, log, dep, grid, c->stream) : arc_trace_launch_f32_hi(a, log, dep, grid, c->stream);
    return a.nb <= 4 ? arc_trace_launch_f64_lo(a, log, dep, grid, c->stream) : arc_trace_launch_f64_hi(a, log, dep, grid, c->stream);
}

cudaError_t arc_launch_pix2vec(const int32_t *d_level, const uint32_t *d_pix, int n, double *d_out, cudaStream_t s)
{
    arc_pix2vec_kernel<<<(n + 127) / 128, 128, 0, s>>>(d_level, d_pix, n, d_out);
    return cudaGetLastError();
}

cudaError_t arc_launch_sched_reset(arc_ctx *c, unsigned long long seed_total)
{
    arc_sched_reset_kernel<<<ARC_QUEUE_CAP / 256, 256, 0, c->stream>>>(c->d_sched, c->d_stats, c->d_qseq, seed_total);
    return cudaGetLastError();
}
