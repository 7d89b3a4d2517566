// arc_internal.cuh -- shared declarations of the CUDA path (not part of the public ABI).
// Nothing here is shared with oracle/: both sides are typed from DESIGN.md's arithmetic contract.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>
#include "../../include/arc.h"

#define ARC_WARPS_PER_BLOCK 8
#define ARC_TRACE_THREADS (32 * ARC_WARPS_PER_BLOCK)
#define ARC_STACK_CAP 512            // families per warp-private stack: <= 32 per level
#define ARC_QUEUE_CAP (1u << 18)     // ring slots of the global donation queue (>> warps x 32 + ARC_QUEUE_LOW)
#define ARC_QUEUE_LOW 4096           // busy warps stop donating above this pool level
#define ARC_BATCH_FAM 8              // families (x4 children = 32 rays) per warp batch

// device-side error codes written to SchedState::error
enum { ARC_DEV_OK = 0, ARC_DEV_STACK_OVERFLOW = 1, ARC_DEV_LOG_OVERFLOW = 2, ARC_DEV_WATCHDOG = 3, ARC_DEV_RAY_RUNAWAY = 4,
       ARC_DEV_CHECK_FAILED = 5 };   // (5: a bounds check of the checked build, -DARC_CHECKED=1: libarc_b200_checked.so)

// The checked build (paper_1807_07094_b200/build.py --checked; tests/test_gpu_checked_build.py runs parity workloads
// through it) verifies, on the device, every index the tracer forms before it is used: cells, sources, levels, ring and
// queue slots, staging addresses, log entries.  compute-sanitizer is not available on the pool this was developed on
// (profiles/r02_sanitizers.md), so the kernel checks itself.  In the normal build ARC_CHECK compiles to nothing.
#ifdef ARC_CHECKED
#define ARC_CHECK(sc_, cond) do { if (!(cond)) atomicCAS(&(sc_)->error, 0, ARC_DEV_CHECK_FAILED); } while (0)
#else
#define ARC_CHECK(sc_, cond) do { } while (0)
#endif

// A "family" = the 4 children 4*fam+j (j = 0..3) of one split (or 4 consecutive root pixels), all at
// `level`, starting at the parent's split radius with the parent's optical depths.  P is the
// photon rate each child still carries, S_nu e^-tau_nu / npix = a quarter of what the parent had left: handing the
// carried value down (instead of re-deriving it from tau) makes emitted = absorbed + escaped hold to rounding
// whatever precision the attenuation factor was evaluated in.
template <int NB>
struct __align__(16) FamRec {
    uint32_t src;
    uint32_t fam;
    uint32_t level;
    uint32_t pad;
    double tau[NB];
    double P[NB];
};

// Every word that idle warps poll or working warps update sits in its own 256-byte block: thousands of idle warps polling
// ONE line keep a single L2 slice saturated (measured: with 3 blocks per SM a lone ray tree ran 2x slower than with 1),
// and the working warps' own scheduler accesses queue up behind the polls.  Spread out, the words hash to different slices.
#ifndef ARC_SCHED_ALIGN
#define ARC_SCHED_ALIGN 256
#endif
struct SchedState {
    alignas(ARC_SCHED_ALIGN) long long in_flight;            // families alive anywhere, as known through flushes
    alignas(ARC_SCHED_ALIGN) unsigned long long seed_next;   // next unclaimed root family
    alignas(ARC_SCHED_ALIGN) unsigned long long q_head;      // donation queue tickets: reserved pops
    alignas(ARC_SCHED_ALIGN) unsigned long long q_tail;      // ... and pushes
    alignas(ARC_SCHED_ALIGN) long long q_count;              // counting semaphore: published - claimed entries (may dip below 0)
    alignas(ARC_SCHED_ALIGN) int hungry;                     // warps idling for work
    alignas(ARC_SCHED_ALIGN) int error;                      // ARC_DEV_*
    alignas(ARC_SCHED_ALIGN) unsigned long long q_high;      // max(q_tail - q_head) seen
    unsigned long long log_n;                                // ray-log entries written
};

struct DevStats {
    unsigned long long segments_total, subcycles_total;     // since arc_create_grid: never reset (arc_run_steps reads them once)
    unsigned long long segments, rays, digest, deposit_records;
    unsigned long long splits[ARC_MAX_LEVEL];
    unsigned long long rays_level[ARC_MAX_LEVEL];
    unsigned long long ends[3];
    double escaped[ARC_MAX_BINS];
    unsigned long long subcycles;
    unsigned int max_sub;
    unsigned int pad;
    unsigned long long chem_next;      // arc_chem_kernel's cell counter (zeroed with the two fields above)
};

// stride (in doubles) of one cell's accumulators: nb rounded up to even (nb > 1) so that a cell's record is a
// multiple of 16 bytes, 16-byte aligned - the granule of cp.reduce.async.bulk
static inline int arc_nbp(int nb) { return nb == 1 ? 1 : ((nb + 1) & ~1); }

struct TraceArgs {
    int N, nb, l0, Lmax, nsrc;
    int NN;                    // N * N (cell stride of a z step)
    unsigned int max_seg;      // 3 N + 8: no ray has more segments (runaway guard)
    int nbp;                   // accumulator stride, arc_nbp(nb)
    double dx;                 // cell size [cm]
    double csplit;             // sqrt(3/(pi Phi)): split radius of level l = csplit * 2^l (cells)
    double tau_term;
    double cpix;               // sqrt(pi/3): pixel width of level l at radius r is r cpix 2^-l (geometric correction)
    int geom;                  // ARC_GEOM_*
    const void *kappa;         // [cell][nb] at field dtype
    double *A;                 // [cell][nbp] absorbed photons/s (entries nb..nbp-1 stay zero)
    const double *src_g;       // [nsrc][3] source position in grid units
    const double *src_S;       // [nsrc][nb] Ndot * binfrac
    const unsigned char *blocked;   // NULL or [nsrc][12 4^l0]: blocked root rays (anisotropic emission)
    // optically thin inner region: all NULL / 0 when off
    double thin_tau;
    const double *Rstart;               // [nsrc] start radius of the root rays (cells)
    unsigned long long *Rnext;          // [nsrc] bits of the radius found by this trace (atomicMin; starts at +inf)
    const unsigned long long *seed_prefix;   // [nsrc + 1] first root family of each source
    const int *src_level;               // [nsrc] level of each source's root rays
    unsigned char *stacks;     // n_warps * ARC_STACK_CAP family records
    unsigned char *queue;      // ARC_QUEUE_CAP family records
    unsigned long long *qseq;  // ARC_QUEUE_CAP slot sequence numbers
    SchedState *sched;
    DevStats *stats;
    unsigned long long seed_total;  // nsrc * 3 * 4^l0
    unsigned int fam_per_src;       // 3 * 4^l0
    int seed_chunk;
    int flags;                      // kernel variant: 1 = per-ray log, 2 = traversal digest
    // ray log (debug)
    unsigned long long *log_key; unsigned int *log_seq; int *log_cell; unsigned long long log_cap;
};

struct Spectrum {
    int nb;
    double E[ARC_MAX_BINS];
    double sig[3][ARC_MAX_BINS];
};

struct arc_ctx {
    int N = 0, dtype = 0;
    int64_t ncell = 0;
    double box_cm = 0, dx = 0;
    arc_params p;
    cudaStream_t stream = 0;
    void *f[5] = {0, 0, 0, 0, 0};     // n_H, x_HI, x_HeI, x_HeII, T at field dtype (SoA)
    Spectrum spec;
    bool have_fields = false, have_spec = false, have_src = false, have_rates = false;
    int nsrc = 0;
    double *d_src_g = 0, *d_src_S = 0;
    std::vector<double> h_src_S;      // host copy of Ndot * binfrac (emitted with an emission mask)
    unsigned char *d_blocked = 0; int mask_level = -1;     // arc_set_emission_mask
    std::vector<double> h_nopen;      // open root rays per source (emission mask), npix0 without a mask
    // optically thin inner region (arc_params.thin_tau > 0): radii found by the last trace, and the device arrays of a trace
    std::vector<double> h_R;
    double *d_Rstart = 0; unsigned long long *d_Rnext = 0; unsigned long long *d_seed_prefix = 0; int *d_src_level = 0;
    double *d_Sopen = 0; int thin_cap = 0;
    double emitted[ARC_MAX_BINS];
    void *d_kappa = 0; int kappa_nb = 0;
    double *d_A = 0; int A_nb = 0;
    double *d_rates = 0;              // 7 * ncell
    unsigned char *d_stacks = 0; size_t stacks_bytes = 0;
    unsigned char *d_queue = 0; unsigned long long *d_qseq = 0; size_t queue_bytes = 0;
    SchedState *d_sched = 0;
    DevStats *d_stats = 0;
    double *d_absorbed = 0;           // [ARC_MAX_BINS] reduction scratch
    unsigned long long *d_dt = 0;     // [2] arc_suggest_dt: min dt (bits of a positive double), cells used
    int n_sm = 0;
    int trace_grid = 0;
    cudaEvent_t ev[8];                // 0..3: trace call (start, after opacity, after kernel, after finalize); 4,7: arc_finalize; 5,6: chemistry
    bool traced_once = false, chem_once = false;
    bool have_accum = false;          // arc_trace_partial ran: the accumulators wait for arc_finalize
    bool finalize_split = false;      // the last finalise pass was arc_finalize's (events 4, 7)
    unsigned long long launches = 0;  // kernels launched by this context (arc_stats.kernel_launches)
    bool queue_dirty = true;          // the donation queue needs its full reset (first trace, or the last one aborted)
    unsigned long long epoch = 0;     // bumped by every call that changes what a captured step graph bakes in
    cudaGraphExec_t step_exec = nullptr; unsigned long long step_epoch = 0; double step_dt = 0.0;   // arc_run_steps
    unsigned long long step_launches = 0;    // kernels in one replay of that graph
    cudaEvent_t ev_steps[2] = {nullptr, nullptr}; bool steps_timed = false;
    bool unchecked = false;           // an asynchronous trace has been enqueued and its device error word not yet looked at
    std::string err;
};

// arc_fields.cu
cudaError_t arc_launch_opacity(arc_ctx *c, unsigned long long seed_total);    // a1 + a2 + the per-trace scheduler / tally reset
cudaError_t arc_launch_finalize(arc_ctx *c);
cudaError_t arc_launch_thin_region(arc_ctx *c, double maxR);     // inner-region deposit for the sources with Rstart > 0
// arc_trace.cu
cudaError_t arc_launch_queue_reset(arc_ctx *c);        // full reset of the donation queue (first trace / after an aborted one)
cudaError_t arc_launch_trace(arc_ctx *c, const TraceArgs &a, bool log, int *grid_out);
int arc_trace_occupancy_grid(arc_ctx *c, int nb, int flags);   // flags: 1 log, 2 digest
cudaError_t arc_launch_pix2vec(const int32_t *d_level, const uint32_t *d_pix, int n, double *d_out, cudaStream_t s);
// arc_run.cu: after the stream has been synchronised - report (and clear) what the last trace left in the device error word
int arc_check_device(arc_ctx *c);
// arc_chem.cu
cudaError_t arc_launch_chemistry(arc_ctx *c, double dt);
cudaError_t arc_launch_suggest_dt(arc_ctx *c, int scheme, double eps);     // result in c->d_dt
