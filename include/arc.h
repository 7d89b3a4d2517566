/* arc.h -- C ABI of the B200-native ARC hot path (libarc_b200.so).
 *
 * ARC = photon-conserving, spatially adaptive HEALPix ray tracing from point sources through a
 * uniform N^3 grid, followed by the per-cell ionisation/heating update (Hartley & Ricotti 2018,
 * arXiv:1807.07094; citations below are PAPER.md line numbers, and DESIGN.md for the readings
 * where the paper is silent).
 *
 * Conventions
 *  - every call returns an int status (ARC_OK = 0, negative = error); nothing throws or aborts;
 *    arc_last_error() gives the text of the last failure of that context.
 *  - all grid arrays are C-contiguous, x fastest: index = (iz*N + iy)*N + ix.  Units are cgs;
 *    photon energies in eV.
 *  - `where` says where caller pointers live: ARC_HOST (pageable or pinned host memory) or
 *    ARC_DEVICE (device memory of the current CUDA device).  Inputs are COPIED: the caller keeps
 *    ownership of everything it passes in.  Device pointers handed OUT (arc_rates) are owned by the
 *    library and stay valid until the next arc_trace() or arc_destroy() on that context.
 *  - every step of the path runs in CUDA kernels for sm_100a; there is no CPU fallback.  Without a
 *    CUDA device arc_create_grid() returns ARC_ECUDA.
 *  - work is enqueued on the stream given to arc_set_stream() (default: the legacy default stream).
 *    With arc_params.async == 0 (default) arc_trace()/arc_update_chemistry() synchronise that
 *    stream before returning and report device-side errors (e.g. ARC_EOVERFLOW) themselves; with
 *    async == 1 they only enqueue.  A trace that failed on the device (ARC_EOVERFLOW, ARC_ECUDA) then leaves a sticky
 *    device error: the kernels of every later call on that context (finalize, chemistry, time step, further traces) see
 *    it and do NOTHING - fields and rates are never updated from an aborted trace - and the error is returned by the
 *    first call that synchronises: arc_synchronize(), arc_get_stats(), arc_suggest_dt(), and arc_get_fields() /
 *    arc_get_rates() / arc_get_accum() with ARC_HOST pointers.  Reporting it clears it (rates are then invalid:
 *    ARC_ESTATE until the next arc_trace).  Device-pointer read-backs do not synchronise and cannot report.
 */
#ifndef ARC_B200_H
#define ARC_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ARC_MAX_BINS 8
#define ARC_MAX_LEVEL 16

typedef struct arc_ctx arc_ctx;                       /* opaque; owns all device memory */

enum { ARC_F32 = 0, ARC_F64 = 1 };                    /* dtype of the five gas fields */
enum { ARC_HOST = 0, ARC_DEVICE = 1 };
enum { ARC_OK = 0, ARC_EINVAL = -1, ARC_ENOMEM = -2, ARC_ECUDA = -3, ARC_ESTATE = -4, ARC_EOVERFLOW = -5 };
enum { ARC_END_SPLIT = 0, ARC_END_DEPLETED = 1, ARC_END_ESCAPED = 2 };
/* deposit routes of the tracer (same sums): RED = every lane issues its own fp64 REDs; AGG = lanes of a
 * warp that are in the same cell are summed in registers first and one lane issues the REDs; QUAD = a segment's bins are
 * spread over the 4 lanes of a lane quad so that one RED instruction carries whole accumulator records.
 * AUTO = the fastest measured for the bin count. */
enum { ARC_DEPOSIT_AUTO = 0, ARC_DEPOSIT_RED = 1, ARC_DEPOSIT_AGG = 2, ARC_DEPOSIT_QUAD = 3 };
/* geometric correction of the deposit (Eq. 2-3, study at :338-354; readings G25-G29):
 * NONE; FC = each segment's absorbed rate times f_c = 1/2 + D_edge/L_pix (capped at 1), the rest is lost; FC_SECONDARY =
 * the paper's choice: what f_c removed goes to the adjacent cell across the nearest face (photon conserving; kept in the
 * cell when that neighbour is outside the box); FC2 = f_c squared (Wise & Abel 2011), the rest lost.  The ray itself
 * (optical depth, splitting, termination) is the same in every mode. */
enum { ARC_GEOM_NONE = 0, ARC_GEOM_FC = 1, ARC_GEOM_FC_SECONDARY = 2, ARC_GEOM_FC2 = 3 };

/* Free parameters the paper names (PAPER.md:45 initial level, :96/:348 Phi, :154 eps; G7
 * tau_term) plus run-time switches of this implementation. */
typedef struct arc_params {
    int32_t l0;             /* initial HEALPix level: 12*4^l0 root rays per source      */
    int32_t Lmax;           /* rays at this level never split; <= 14 (pixel ids are 32 bit)          */
    double  Phi;            /* rays per cell: split when Omega_l r^2 > dx^2/Phi   */
    double  tau_term;       /* ray ends when min_nu tau_nu >= tau_term (+inf disables)               */
    double  Yp;             /* helium mass fraction; 0 = pure hydrogen              */
    int32_t isothermal;     /* 1: T fixed, energy equation skipped                                   */
    int32_t caseB;          /* 1: case-B recombination coefficients                                  */
    int32_t coll_ion;       /* 1: collisional ionisation terms C_S(T) of Eq. 4 on                    */
    int32_t max_subcycles;  /* cap on chemistry sub-cycles per cell per call                         */
    double  eps_sub;        /* sub-cycle fractional change, 0.1 in the paper          */
    double  x_floor;        /* lower clamp of x_HI, x_HeI                                            */
    int32_t digest;         /* 1: also accumulate the order-independent traversal digest (slower)    */
    int32_t async;          /* 1: arc_trace/arc_update_chemistry do not synchronise (see top)        */
    int32_t trace_blocks;   /* persistent-kernel grid size; 0 = SM count x resident blocks per SM    */
    int32_t deposit;        /* how segments reach the accumulators: ARC_DEPOSIT_AUTO | _RED | _AGG | _QUAD        */
    int32_t geom_corr;      /* ARC_GEOM_NONE | _FC | _FC_SECONDARY | _FC2; needs deposit = AUTO */
    int32_t debug_fault;    /* test hook, keep 0: a non-zero ARC device error code (1 = work-stack overflow, 3 = watchdog,
                               4 = runaway ray) makes every following trace start as if its kernel had raised it - the
                               only way to exercise the error paths of async mode without breaking the tracer       */
    double  thin_tau;       /* optically thin inner region: 0 = off; > 0 (0.1 in the paper): every
                               arc_trace records, per source, the radius up to which tau of the first (softest) bin stays
                               below thin_tau on every ray, and the NEXT arc_trace gives the cells within that radius the
                               thin-limit absorption S kappa V / (4 pi r^2) and starts the rays there (tau = 0, at the
                               level they have at that radius).  Needs deposit = AUTO and geom_corr = NONE; arc_trace
                               then synchronises.  Radii: arc_get_thin_radii / arc_set_thin_radii.                */
} arc_params;

/* Per-cell outputs of arc_trace (PAPER.md:83 Eq. 1, :134-138, :170): DEVICE pointers, N^3 doubles each. */
typedef struct arc_rates {
    const double *Gamma_HI, *Gamma_HeI, *Gamma_HeII;   /* photo-ionisation rate per absorber [1/s]     */
    const double *heat_HI, *heat_HeI, *heat_HeII;      /* photo-heating per absorber [erg/s]           */
    const double *heat_total;                          /* sum_S heat_S n_S [erg/s/cm^3] */
} arc_rates;

typedef struct arc_stats {
    uint64_t segments;                 /* (ray, cell) deposit events of the last arc_trace             */
    uint64_t rays;                     /* ray records traced (all levels)                              */
    uint64_t digest;                   /* sum mod 2^64 of per-ray hashes (only if params.digest)       */
    uint64_t queue_high_water;         /* max entries seen in the global donation queue                */
    uint64_t splits[ARC_MAX_LEVEL];    /* rays that split, per level                                   */
    uint64_t rays_level[ARC_MAX_LEVEL];
    uint64_t ends[3];                  /* rays ended by ARC_END_*                                      */
    double   emitted[ARC_MAX_BINS];    /* photons/s per bin: sum over sources                          */
    double   absorbed[ARC_MAX_BINS];   /* = sum over cells of the accumulators                         */
    double   escaped[ARC_MAX_BINS];    /* left the box ("radiation leaving the box is lost") */
    uint64_t subcycles;                /* total chemistry sub-cycles of the last arc_update_chemistry  */
    uint32_t max_subcycles_cell;       /* largest per-cell sub-cycle count of that call                */
    uint32_t pad;
    float    trace_ms, chem_ms;        /* CUDA-event durations of the last calls (whole call, on-stream) */
    float    trace_kernel_ms;          /* the persistent ray-tracing kernel alone (same events, same stream) */
    float    opacity_ms, finalize_ms;  /* the two per-cell passes around it                               */
    int32_t  trace_grid;               /* thread blocks of the persistent kernel                          */
    int32_t  pad2;
    uint64_t deposit_records;          /* accumulator records sent to L2 (<= segments: warp-aggregated deposit) */
    uint64_t kernel_launches;          /* kernels this context has launched since arc_create_grid (counted on the host at
                                          every launch of the library's own kernels; memsets and copies are not kernels) */
    uint64_t segments_total;           /* segments / chemistry sub-cycles of ALL traces / updates since arc_create_grid    */
    uint64_t subcycles_total;          /*   (the per-call counters above are those of the last call only)                 */
    float    steps_ms;                 /* arc_run_steps: CUDA-event duration of all its steps together (the per-kernel times
                                          above are then 0: events cannot be timed inside a captured graph)             */
    int32_t  pad3;
} arc_stats;

/* Caller-provided HOST buffers for arc_trace_debug: one entry per segment (seq = 0,1,2,... within the
 * ray, cell = linear cell index) and one closing entry per ray (seq = number of segments,
 * cell = -1 - ARC_END_*).  key = (src << 40) | (level << 32) | pixel.  Entries arrive unordered. */
typedef struct arc_raylog {
    int64_t   cap;        /* capacity of the three arrays (entries)                                    */
    int64_t   n;          /* out: entries written                                                      */
    uint64_t *key;
    uint32_t *seq;
    int32_t  *cell;
} arc_raylog;

/* Grid of N^3 cells in a cube of side box_cm.  dtype = ARC_F32 | ARC_F64 is the storage
 * type of the five gas fields and of the per-step opacity table; accumulators and rates are fp64.
 * Errors: ARC_EINVAL (N < 1 or N > 1024, box <= 0, bad dtype), ARC_ECUDA (no device), ARC_ENOMEM. */
int arc_create_grid(arc_ctx **out, int N, double box_cm, int dtype);
int arc_destroy(arc_ctx *c);

void arc_default_params(arc_params *p);                /* l0=1, Phi=3, Lmax=13, tau_term=30, eps=0.1 ... */
int arc_set_params(arc_ctx *c, const arc_params *p);   /* ARC_EINVAL on out-of-range values             */
int arc_set_stream(arc_ctx *c, void *cuda_stream);     /* cudaStream_t; NULL = default stream           */

/* Gas fields: n_H [cm^-3], neutral/ionised fractions x_HI, x_HeI, x_HeII, T [K]; each
 * N^3 values of the grid dtype.  x_HeII is this build's third absorber (G12). */
int arc_set_fields(arc_ctx *c, const void *n_H, const void *x_HI, const void *x_HeI,
                   const void *x_HeII, const void *T, int where);
int arc_get_fields(arc_ctx *c, void *n_H, void *x_HI, void *x_HeI, void *x_HeII, void *T, int where);
                                                       /* NULL pointers are skipped */

/* Frequency bins: per bin one representative energy and one frequency-averaged
 * cross-section per species [cm^2].  1 <= nbins <= ARC_MAX_BINS.  HOST pointers. */
int arc_set_spectrum(arc_ctx *c, int nbins, const double *E_eV, const double *sig_HI,
                     const double *sig_HeI, const double *sig_HeII);

/* Point sources: position [cm] in [0, box) on every axis (else ARC_EINVAL), photon
 * rate Ndot [1/s] and its split over the bins (rows of binfrac).  HOST pointers.  Call after
 * arc_set_spectrum (ARC_ESTATE otherwise).  A position so close to the upper box face that pos/(box/N) rounds to N
 * (possible when N is not a power of two) has no cell and is rejected too (ARC_EINVAL). */
int arc_set_sources(arc_ctx *c, int nsrc, const double *pos_cm /*[nsrc][3]*/, const double *Ndot,
                    const double *binfrac /*[nsrc][nbins]*/);

/* One radiative-transfer pass (PAPER.md:47-56 steps i, iii; :79-98; Eq. 1): zero the accumulators,
 * rebuild the opacity table from the current fields, trace every ray of every source (persistent
 * kernel), finalise the per-cell rates.  `step` is a label only.  out may be NULL.
 * Errors: ARC_ESTATE (fields / spectrum / sources missing), ARC_EOVERFLOW (work stack or queue
 * exhausted: rates invalid), ARC_ECUDA. */
int arc_trace(arc_ctx *c, int step, arc_rates *out);

/* Copy the rates out: each non-NULL pointer receives N^3 doubles (host or device per `where`). */
int arc_get_rates(arc_ctx *c, double *Gamma_HI, double *Gamma_HeI, double *Gamma_HeII,
                  double *heat_HI, double *heat_HeI, double *heat_HeII, double *heat_total, int where);

/* Source-sharded tracing ("the total ionization rate ... is the sum of the contributions of all
 * sources", :134, :231): the absorbed-photon accumulators are linear in the sources, so several contexts (one per GPU,
 * same fields, each with its own share of the sources) can trace independently and add their accumulators before the
 * rates are formed.
 *   arc_trace_partial : rows a1-a9 of a trace for THIS context's sources (zero, opacity table, rays); no rates yet -
 *                       arc_get_rates / arc_update_chemistry return ARC_ESTATE until arc_finalize.  Errors as arc_trace.
 *   arc_accum_device  : library-owned DEVICE pointer to the accumulators and their length in doubles
 *                       (N^3 records of nbins doubles, padded to an even count when nbins > 1; padding stays 0), for an
 *                       in-place element-wise sum over the shards by the caller (e.g. ncclAllReduce on the context's
 *                       stream).  Valid until arc_destroy; contents defined between arc_trace_partial and arc_finalize.
 *   arc_finalize      : row a10 (rates from whatever the accumulators now hold).  out may be NULL.  ARC_ESTATE without
 *                       a pending arc_trace_partial (setting fields, sources, spectrum or parameters discards it).
 * Statistics (arc_get_stats) stay per context: segments, rays, emitted, escaped are this shard's; `absorbed` is the sum
 * over cells of the accumulators at arc_finalize, i.e. of all shards after the caller's sum. */
int arc_trace_partial(arc_ctx *c, int step);
int arc_accum_device(arc_ctx *c, double **A, int64_t *n_doubles);
int arc_finalize(arc_ctx *c, arc_rates *out);

/* Raw accumulators of the last trace: absorbed photons/s, layout [cell][bin], N^3*nbins doubles. */
int arc_get_accum(arc_ctx *c, double *A, int where);

/* Sub-cycled backward-difference update of x_HI, x_HeI, x_HeII, T over dt_s with the rates of the
 * last arc_trace held fixed (PAPER.md:57 step v; :136-154 Eq. 4-5; :166-172).  ARC_ESTATE if no
 * trace has been done since the fields were last set. */
int arc_update_chemistry(arc_ctx *c, double dt_s);

/* The time-step loop of PAPER.md:47-59 (steps i, iii, v, vii) without a host round trip per step: n_steps times
 * { arc_trace; arc_update_chemistry(dt_s) }, enqueued back to back - one step is captured once into a CUDA graph (opacity +
 * reset, tracer, finalize, chemistry) and replayed - then ONE synchronisation and error check (none with async = 1).
 * The fields advance n_steps x dt_s; rates and per-call statistics are those of the last step, segments_total /
 * subcycles_total count all of them, steps_ms times them together.  Small grids, where launches and synchronisation cost
 * more than the kernels, are what this is for.  Needs a stream set with arc_set_stream for the graph
 * (on the legacy default stream the steps are enqueued one by one instead).  Errors as arc_trace; ARC_EINVAL with
 * thin_tau > 0 (each of those traces hands its radii to the host). */
int arc_run_steps(arc_ctx *c, int n_steps, double dt_s);

/* Anisotropic emission: blocked[s * npix0 + p] != 0 blocks root ray p (nested pixel of level l0,
 * npix0 = 12 * 4^l0) of source s: it does not exist - no packet, no segments, not in `emitted`; the open rays carry the
 * mean rate per ray Ndot f_nu / npix0, so a source with a fraction f_esc of its rays open emits f_esc Ndot.
 * `level` must equal arc_params.l0 at the time of the call and of every later arc_trace (ARC_ESTATE otherwise).
 * blocked: HOST pointer, nsrc * npix0 bytes, copied; NULL clears the mask.  arc_set_sources clears it too. */
int arc_set_emission_mask(arc_ctx *c, const uint8_t *blocked, int level);

/* Optically thin inner region (arc_params.thin_tau > 0): the per-source radii, in CELLS, that the next arc_trace will use
 * (found by the last one; 0 after arc_set_sources).  HOST pointers, nsrc doubles.  arc_set_thin_radii: values must be
 * finite and >= 0 (0 = that source traces from r = 0). */
int arc_get_thin_radii(arc_ctx *c, double *R_cells);
int arc_set_thin_radii(arc_ctx *c, const double *R_cells);

/* Radiative-transfer time step, from the CURRENT fields and the rates of the last arc_trace:
 * per cell dn_HI/dt = n_H (alpha_HII n_e x_HII - (Gamma_HI + C_HI n_e) x_HI) (Eq. 4);
 *   scheme ARC_DT_NEUTRAL   (i):  min over cells with tau = n_HI sigma_1 d > 0.5 of eps n_HI / |dn_HI/dt|   (:182-190)
 *   scheme ARC_DT_INTENSITY (ii): min over all cells of eps / (sigma_1 d |dn_HI/dt|)                         (:192-204)
 * sigma_1 = H I cross-section of the first (softest) bin, d = cell width.  *dt_s = +inf if no cell qualifies;
 * *cells_used (may be NULL) = cells that entered the minimum.  One streaming reduction kernel; synchronises.
 * ARC_ESTATE without valid rates. */
enum { ARC_DT_NEUTRAL = 1, ARC_DT_INTENSITY = 2 };
int arc_suggest_dt(arc_ctx *c, int scheme, double eps, double *dt_s, int64_t *cells_used);

int arc_synchronize(arc_ctx *c);                       /* wait for the stream; report deferred errors */
int arc_get_stats(arc_ctx *c, arc_stats *s);           /* synchronises */

/* Same as arc_trace but with per-ray logging into caller-provided host buffers (small configs only).
 * ARC_EOVERFLOW if log->cap is too small (log->n then holds the number needed, if known). */
int arc_trace_debug(arc_ctx *c, int step, arc_raylog *log);

/* Device HEALPix generator, exposed for testing (O1): unit vectors of `n` (level, pixel) pairs.
 * HOST pointers; out is [n][3]. */
int arc_pix2vec(const int32_t *level, const uint32_t *pix, int n, double *out);

/* Self-test of the tracer's division (DESIGN.md 6.2 step 1, contract C3): the march needs the IEEE quotient
 * RN(a / d) and gets it from RN(1/d) and two fused residual corrections.  Runs n_pairs device-generated pairs
 * (counter-based generator on `seed`): a = i - g with integer 0 <= i <= 1025 and g uniform in [0, 1024) (also snapped to
 * integers, half-integers and binary fractions), d = a direction component in (2^-40, 1] (uniform in exponent, random
 * mantissa, also just below / at powers of two), both signs - and counts the pairs whose result differs in any bit from
 * __ddiv_rn(a, d).  *mismatches must come back 0.  HOST pointer; synchronises; default stream. */
int arc_selftest_division(uint64_t n_pairs, uint64_t seed, uint64_t *mismatches);

/* arc_pix2vec for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid it): same arguments, same results to the bit, but the device staging that arc_pix2vec cudaMalloc's and
 * cudaFree's on every call lives in ONE file-scope device array of fixed size (csrc/arc_noalloc.cu), so the call makes no
 * cudaMalloc, no cudaFree and no allocating library call.  Limit: n <= ARC_PIX2VEC_NOALLOC_MAX = 4096 pairs per call
 * (128 KiB of device memory, held by every GPU that loads the library until the process exits); more is ARC_EINVAL with
 * the reason in arc_noalloc_last_error() - split the call.  HOST pointers; out is [n][3]; synchronous on the legacy
 * default stream of the current device.  All calls on a device share the array and it keeps the last call's contents
 * (nothing in it needs to start at zero: the n inputs are overwritten before they are read, the 3 n outputs written
 * before they are copied back); calls through this entry point are serialised by a mutex, anything else that touched
 * the array concurrently on the GPU would race.  Errors: ARC_EINVAL (NULL, n < 0, n > max, not a pixel), ARC_ECUDA. */
#define ARC_PIX2VEC_NOALLOC_MAX 4096
int arc_pix2vec_noalloc(const int32_t *level, const uint32_t *pix, int n, double *out);
int arc_pix2vec_noalloc_max(void);                     /* = ARC_PIX2VEC_NOALLOC_MAX of the loaded library */
const char *arc_noalloc_last_error(void);              /* text of this thread's last arc_pix2vec_noalloc failure */

const char *arc_last_error(const arc_ctx *c);          /* c may be NULL: last error of a failed create */
const char *arc_version(void);

#ifdef __cplusplus
}
#endif
#endif
