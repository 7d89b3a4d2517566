// arc_trace_kernel.cuh -- the persistent ray-tracing kernel, as a template that the
// arc_trace_inst_*.cu translation units instantiate (split so that they compile in parallel).
//
// What it computes (Eq. 1; O1-O3): every source emits 12*4^l0 HEALPix
// rays; a ray marches cell by cell (3D-DDA: next X, Y or Z boundary), each segment adds
// S_nu e^-tau_nu (1 - e^-dtau_nu) absorbed photons/s to the cell's accumulator (atomically),
// and at radius r_split(l) = sqrt(3/(pi Phi)) 2^l cells the ray is replaced by its 4 HEALPix children.
//
// How (B200 design, NOT the paper's per-source, per-level launches - PAPER.md:49-54 is prior art):
//  * ONE launch for all sources and all levels.  The grid is sized to what is co-resident
//    (SMs x blocks/SM); every warp runs a work loop until a global in-flight counter reaches zero.
//  * Work item = a FAMILY (4 sibling rays sharing start radius and optical depths), so a split costs one
//    record; 8 families = one warp batch; lane = (family, child).  Siblings/neighbouring pixels sit in
//    neighbouring lanes (nested order), which keeps opacity gathers and atomics on neighbouring cells.
//  * Each warp owns a LIFO stack in global memory (depth-first => bounded memory: <= 32 families per
//    level).  Survivors of a batch are compacted with a ballot/popc prefix and pushed in one step.
//  * Load balance: root families come from a global seed counter; idle warps raise `hungry` and busy
//    warps keep their next batch and donate the rest of their stack, shallow end first (biggest subtrees),
//    through a bounded MPMC ticket queue; idle warps take whole batches once the trace is deep.
//  * Deposit: fire-and-forget fp64 REDs into the cell's accumulator record.  The RED path costs
//    per LANE (one L1 wavefront / L2 sector op each), so lanes of a warp that are in the same cell in the same
//    iteration - siblings and neighbouring pixels run almost parallel less than a cell apart - are first summed
//    in registers (match.any on the cell index, shuffles) and one lane issues the REDs for the group.
//  * Deterministic arithmetic (contract C0-C5): every operation that decides a cell, an axis, a split or a
//    termination is an explicit IEEE round-to-nearest intrinsic (no FMA contraction), typed from DESIGN.md.
#pragma once
#include "arc_internal.cuh"
#include "arc_healpix.cuh"
#include "arc_divide.cuh"

#define FLAG_LOG 1          // template flag: per-ray logging (arc_trace_debug)
#define FLAG_DIGEST 2       // template flag: accumulate the order-independent traversal digest
#define FLAG_GEOM 4         // template flag: geometric correction of the deposit (Eq. 2-3), mode in TraceArgs::geom
#ifndef ARC_GREEDY_MIN_INFLIGHT
#define ARC_GREEDY_MIN_INFLIGHT 2048   // families alive above which idle warps take whole batches from the donation queue
#endif
#ifndef ARC_DONATE_KEEP
#define ARC_DONATE_KEEP 8              // a donor keeps its next batch (8 families) and gives away the rest, 32 at a time
#endif
#ifndef ARC_POOL_PER_HUNGRY
#define ARC_POOL_PER_HUNGRY ARC_BATCH_FAM      // donors keep the pool at this many families per idle warp
#endif
#define FLAG_THIN 8         // template flag: track, per source, the radius up to which tau (bin 0) stays below thin_tau

#ifndef ARC_GEOM_MIN_BLOCKS
#define ARC_GEOM_MIN_BLOCKS 3      // ... of the variants with the geometric correction (measured: 2 blocks / 128 registers / no spills
#endif                             // 56.4 G segments/s on config 4, 3 blocks / 80 registers / 200 B of spills 57.3: issue bound either way)
#ifndef ARC_TRACE_MIN_BLOCKS
#define ARC_TRACE_MIN_BLOCKS 3     // resident blocks per SM the register budget is held to (<= 85 registers)
#endif
#define DEP_RED 1           // every lane: nb fp64 REDs per segment
#define DEP_AGG 2           // lanes of a warp that sit in the same cell are summed first (match.any + shuffles): one lane REDs
#define DEP_T 3             // transposed: a cell's bins are spread over the 4 lanes of a lane quad (through shared memory), so
                            // that ONE RED instruction carries whole accumulator records (L1 coalesces the quad's 4 doubles)

namespace {

__device__ __forceinline__ unsigned long long mix64(unsigned long long x)   // splitmix64 finaliser
{
    x ^= x >> 30; x *= 0xbf58476d1ce4e5b9ull;
    x ^= x >> 27; x *= 0x94d049bb133111ebull;
    x ^= x >> 31;
    return x;
}

__device__ __forceinline__ unsigned long long ld_volatile_u64(const unsigned long long *p)
{
    return *(const volatile unsigned long long *)p;
}
__device__ __forceinline__ long long ld_volatile_s64(const long long *p) { return *(const volatile long long *)p; }
__device__ __forceinline__ int ld_volatile_s32(const int *p) { return *(const volatile int *)p; }

__device__ __forceinline__ unsigned long long globaltimer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    return t;
}

// fire-and-forget fp64 reduction (REDG.E.ADD.F64): written as PTX `red` because ptxas otherwise emits the returning
// form (ATOMG ... RZ) inside this kernel's divergent loop, which holds a scoreboard until L2 answers
__device__ __forceinline__ void arc_red_add(double *p, double v)
{
    asm volatile("red.relaxed.gpu.global.add.f64 [%0], %1;" ::"l"(p), "d"(v) : "memory");
}

// the same under a predicate (@p REDG: no branch, no reconvergence barrier around it)
__device__ __forceinline__ void arc_red_add_if(double *p, double v, bool take)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.s32 p, %2, 0;\n\t@p red.relaxed.gpu.global.add.f64 [%0], %1;\n\t}" ::"l"(p), "d"(v), "r"((int)take) : "memory");
}

// opacity gather: the NB opacities of one cell, kept at their storage type until used (fewer registers while
// the prefetched copy is in flight); one vector load per cell where the layout allows
template <typename KT, int NB> struct KVec;
template <int NB> struct KVec<float, NB> {
    float k[NB];
    __device__ __forceinline__ void load(const float *base, int cell)
    {
        const float *p = base + (long long)cell * NB;
        if constexpr (NB % 4 == 0) {
#pragma unroll
            for (int v = 0; v < NB; v += 4) { const float4 q = __ldg((const float4 *)(p + v)); k[v] = q.x; k[v + 1] = q.y; k[v + 2] = q.z; k[v + 3] = q.w; }
        } else if constexpr (NB % 2 == 0) {
#pragma unroll
            for (int v = 0; v < NB; v += 2) { const float2 q = __ldg((const float2 *)(p + v)); k[v] = q.x; k[v + 1] = q.y; }
        } else {
#pragma unroll
            for (int v = 0; v < NB; ++v) k[v] = __ldg(p + v);
        }
    }
    __device__ __forceinline__ double get(int v) const { return (double)k[v]; }
};
template <int NB> struct KVec<double, NB> {
    double k[NB];
    __device__ __forceinline__ void load(const double *base, int cell)
    {
        const double *p = base + (long long)cell * NB;
        if constexpr (NB % 2 == 0) {
#pragma unroll
            for (int v = 0; v < NB; v += 2) { const double2 q = __ldg((const double2 *)(p + v)); k[v] = q.x; k[v + 1] = q.y; }
        } else {
#pragma unroll
            for (int v = 0; v < NB; ++v) k[v] = __ldg(p + v);
        }
    }
    __device__ __forceinline__ double get(int v) const { return k[v]; }
};

// E = e^-x and ome = 1 - e^-x for x >= 0, both to ~2e-14 relative - ome also for tiny x, where 1 - E would
// cancel.  Not a decision: terminations are decided on tau (sums and products only, contract C4).
// x = -(k ln2 + r) with |r| <= ln2/2;  e^r - 1 = r q(r),  q(r) = sum_{n=0..10} r^n/(n+1)!
__device__ __forceinline__ void arc_attenuate(double x, double &E, double &ome)
{
    const double MAGIC = 6755399441055744.0;                           // 1.5 * 2^52: round to nearest integer
    const double kt = fma(x, -1.4426950408889634074, MAGIC);
    const int k = __double2loint(kt);
    const double kd = kt - MAGIC;
    double r = fma(kd, -6.93147180369123816490e-01, -x);               // ln2 split in two parts
    r = fma(kd, -1.90821492927058770002e-10, r);
    double q = 1.0 / 39916800.0;
    q = fma(q, r, 1.0 / 3628800.0);
    q = fma(q, r, 1.0 / 362880.0);
    q = fma(q, r, 1.0 / 40320.0);
    q = fma(q, r, 1.0 / 5040.0);
    q = fma(q, r, 1.0 / 720.0);
    q = fma(q, r, 1.0 / 120.0);
    q = fma(q, r, 1.0 / 24.0);
    q = fma(q, r, 1.0 / 6.0);
    q = fma(q, r, 0.5);
    q = fma(q, r, 1.0);
    const double em1 = r * q;                                          // e^r - 1
    const double scale = __hiloint2double((max(k, -1022) + 1023) << 20, 0);    // 2^k
    const double Ek = (x < 708.0) ? fma(em1, scale, scale) : 0.0;
    E = Ek;
    ome = (k == 0) ? -em1 : 1.0 - Ek;
}

// x += o under a predicate: one predicated DADD (the compiler's own choice is DADD + two selects)
__device__ __forceinline__ void arc_add_if(double &x, double o, int take)
{
    asm("{\n\t.reg .pred p;\n\tsetp.ne.s32 p, %2, 0;\n\t@p add.rn.f64 %0, %0, %1;\n\t}" : "+d"(x) : "d"(o), "r"(take));
}

// two fp32 lanes per instruction (FMUL2 / FFMA2 on sm_100)
__device__ __forceinline__ unsigned long long arc_pack2(float lo, float hi)
{
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void arc_unpack2(unsigned long long r, float &lo, float &hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(r));
}
__device__ __forceinline__ unsigned long long arc_mul2(unsigned long long a, unsigned long long b)
{
    unsigned long long r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ unsigned long long arc_fma2(unsigned long long a, unsigned long long b, unsigned long long c)
{
    unsigned long long r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}

// 2^y for y <= 0 on the SFU (ex2.approx.ftz: ~2 ulp, flushes to zero below 2^-126 - exactly what an attenuation
// factor wants)
__device__ __forceinline__ float arc_ex2(float y)
{
    float r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(y));
    return r;
}

// ---------------------------------------------------------------------------------------------------
template <int NB, typename KT, int FLAGS, int DEP>
__global__ void __launch_bounds__(ARC_TRACE_THREADS, (FLAGS & FLAG_GEOM) ? ARC_GEOM_MIN_BLOCKS : ARC_TRACE_MIN_BLOCKS) arc_trace_kernel(const TraceArgs a)
{
    typedef FamRec<NB> Rec;
    const int lane = threadIdx.x & 31;
    const int gwarp = blockIdx.x * ARC_WARPS_PER_BLOCK + (threadIdx.x >> 5);
    Rec *const stack = reinterpret_cast<Rec *>(a.stacks) + (size_t)gwarp * ARC_STACK_CAP;
    Rec *const queue = reinterpret_cast<Rec *>(a.queue);
    SchedState *const sc = a.sched;
    const KT *const kappa = reinterpret_cast<const KT *>(a.kappa);
    const int N = a.N;
    constexpr int NBP = (NB == 1) ? 1 : ((NB + 1) & ~1);      // accumulator record stride (arc_nbp)
    constexpr int NBE = (NB + 1) & ~1;                        // bins rounded up to whole fp32 pairs
    unsigned long long nred = 0;                              // deposit records this lane sent to L2

    // per-block tallies: 32-bit shared atomics are native (64-bit ones are CAS loops); added to the 64-bit global
    // counters at the end.  A block traces < 2^32 rays: at most 1.2e7 rays per source and 2^24 sources spread over
    // >= 148 blocks would be needed to wrap one, i.e. > 5e12 rays = weeks of tracing in one launch.
    __shared__ unsigned int s_splits[ARC_MAX_LEVEL], s_rays[ARC_MAX_LEVEL], s_ends[3];
    __shared__ double s_esc[ARC_MAX_BINS];
    __shared__ double s_geo[9][ARC_TRACE_THREADS];            // per thread: source position g[3], direction d[3], RN(1/d)[3]
    // DEP_T staging, per warp: NB planes of 32 doubles (plane = bin, column = lane), planes 33 doubles apart.  A lane
    // stores its NB absorbed rates with NB 64-bit stores (consecutive lanes, consecutive words: conflict free); in pass k
    // lane (quad q, b) reads column 4q + k of plane b: word 33 b + 4 q + k, i.e. bank pairs 2b + 8q (+ const) - all 16
    // lanes of a half warp distinct.  Addresses are kept as two opaque registers (else ptxas re-derives them from
    // %tid every iteration); bins and passes are immediate offsets.
    constexpr int DEP_PLANE = 33 * 8;                         // bytes between planes
    constexpr int DEP_WARP = ((NB * DEP_PLANE + 255) / 256) * 256;     // 256-aligned warp regions: (dep_wr >> 3) & 31 is the lane
    __shared__ __align__(256) unsigned char s_dep[DEP == DEP_T ? ARC_WARPS_PER_BLOCK * DEP_WARP : 16];
    [[maybe_unused]] unsigned dep_wr = 0, dep_rd = 0;         // shared-memory byte addresses: my column of plane 0 / column 4q of plane b
    if constexpr (DEP == DEP_T) {
        const unsigned base = (unsigned)__cvta_generic_to_shared(s_dep) + (threadIdx.x >> 5) * DEP_WARP;
        dep_wr = base + (unsigned)lane * 8u;
        dep_rd = base + (unsigned)(lane & 3) * DEP_PLANE + (unsigned)(lane >> 2) * 32u;
        asm volatile("" : "+r"(dep_wr), "+r"(dep_rd));
    }
    // shared-memory byte address of s_geo[0][threadIdx.x] (opaque for the same reason); row stride ARC_TRACE_THREADS * 8
    unsigned geo_ad = (unsigned)__cvta_generic_to_shared(&s_geo[0][threadIdx.x]);
    asm volatile("" : "+r"(geo_ad));
    if (threadIdx.x < ARC_MAX_LEVEL) { s_splits[threadIdx.x] = 0; s_rays[threadIdx.x] = 0; }
    if (threadIdx.x < 3) s_ends[threadIdx.x] = 0;
    if (threadIdx.x < ARC_MAX_BINS) s_esc[threadIdx.x] = 0.0;
    // a sticky device error from an earlier asynchronous trace (or arc_params.debug_fault): this trace does not run; its
    // root families stay "in flight", which tells every consumer kernel to skip (block-uniform decision)
    __shared__ int s_abort;
    if (threadIdx.x == 0) s_abort = ld_volatile_s32(&sc->error);
    __syncthreads();
    if (s_abort != 0) return;

    // own stack = ring of ARC_STACK_CAP records holding families [bot, top) (monotonic counters, warp-uniform)
    unsigned bot = 0, top = 0;
#define STK(i) stack[(i) & (ARC_STACK_CAP - 1)]
    long long delta = 0;                  // families created - consumed since the last flush (warp-uniform)
    unsigned long long nseg = 0, digest = 0;
    bool registered_hungry = false;
    bool quit = false;

    while (!quit) {
        // ------------------------------------------------------------------ acquire work
        if (top == bot) {
            if (delta != 0) { if (lane == 0) atomicAdd((unsigned long long *)&sc->in_flight, (unsigned long long)delta); delta = 0; }
            unsigned long long t_idle0 = 0; long long last_seen = 0; unsigned backoff = 64;
            for (;;) {
                // (1) donated families: claim up to `want` published entries from the counting semaphore
                // q_count, then take that many consecutive tickets.  No retry loops: every atomic succeeds.
                int n = 0; unsigned long long ticket = 0;
                if (lane == 0) {
                    const long long avail = ld_volatile_s64(&sc->q_count);
                    if (avail > 0) {
                        // How much to take.  A warp iteration costs the same with 4 lanes busy as with 32, so once a trace has
                        // deep levels alive (many families in flight: long rays) a whole batch per warp beats one family per
                        // idle warp.  While few families exist (start of a trace, tiny traces: short rays, the queue hop is
                        // what costs) an equal share per idle warp spreads the tree fastest.  Measured, DESIGN.md 6.2.
                        long long want;
                        if (ld_volatile_s64(&sc->in_flight) >= ARC_GREEDY_MIN_INFLIGHT) want = min((long long)ARC_BATCH_FAM, avail);
                        else {
                            const int hungry_now = max(ld_volatile_s32(&sc->hungry), 1);
                            want = max(1ll, min((long long)ARC_BATCH_FAM, avail / hungry_now));
                        }
                        const long long before = (long long)atomicAdd((unsigned long long *)&sc->q_count, (unsigned long long)(-want));
                        const long long got = max(0ll, min(before, want));
                        if (got < want) atomicAdd((unsigned long long *)&sc->q_count, (unsigned long long)(want - got));
                        if (got > 0) { ticket = atomicAdd(&sc->q_head, (unsigned long long)got); n = (int)got; }
                    }
                }
                n = __shfl_sync(0xffffffffu, n, 0);
                ticket = __shfl_sync(0xffffffffu, ticket, 0);
                if (n > 0) {
                    if (lane < n) {
                        const unsigned long long tk = ticket + lane;
                        const unsigned slot = (unsigned)(tk % ARC_QUEUE_CAP);
                        ARC_CHECK(sc, top + lane - bot < ARC_STACK_CAP);
                        while (ld_volatile_u64(&a.qseq[slot]) != tk + 1) __nanosleep(32);
                        __threadfence();
                        const int4 *src = reinterpret_cast<const int4 *>(&queue[slot]);
                        int4 *dst = reinterpret_cast<int4 *>(&STK(top + lane));
#pragma unroll
                        for (int w = 0; w < (int)(sizeof(Rec) / 16); ++w) dst[w] = __ldcg(src + w);
                        __threadfence();
                        *(volatile unsigned long long *)&a.qseq[slot] = tk + ARC_QUEUE_CAP;   // slot free for the next lap
                    }
                    top += n;
                    break;
                }
                // (2) root families (a3: r = 0, tau = 0)
                unsigned long long s0 = 0;
                if (lane == 0 && ld_volatile_u64(&sc->seed_next) < a.seed_total) {
                    s0 = atomicAdd(&sc->seed_next, (unsigned long long)a.seed_chunk);
                    if (s0 < a.seed_total) n = (int)min((unsigned long long)a.seed_chunk, a.seed_total - s0);
                }
                n = __shfl_sync(0xffffffffu, n, 0);
                s0 = __shfl_sync(0xffffffffu, s0, 0);
                if (n > 0) {
                    if (lane < n) {
                        Rec r;
                        const unsigned long long s = s0 + lane;
                        if (a.seed_prefix == nullptr) {
                            r.src = (uint32_t)(s / a.fam_per_src); r.fam = (uint32_t)(s % a.fam_per_src);
                            r.level = (uint32_t)a.l0;
                        } else {
                            // optically thin start (PAPER.md:130 (iv)): source i owns root families [prefix[i], prefix[i+1]) at its
                            // own level src_level[i]; binary search for the source
                            int lo = 0, hi = a.nsrc;                      // prefix[lo] <= s < prefix[hi]
                            while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (__ldg(a.seed_prefix + mid) <= s) lo = mid; else hi = mid; }
                            r.src = (uint32_t)lo; r.fam = (uint32_t)(s - __ldg(a.seed_prefix + lo));
                            r.level = (uint32_t)__ldg(a.src_level + lo);
                        }
                        ARC_CHECK(sc, r.src < (uint32_t)a.nsrc && r.level <= (uint32_t)a.Lmax && r.fam < (3u << (2 * r.level)) && top + lane - bot < ARC_STACK_CAP);
                        r.pad = 1;                                        // root family: starts at Rstart[src] (0 without a thin region)
                        const double npix0 = (double)(12ull << (2 * r.level));
#pragma unroll
                        for (int v = 0; v < NB; ++v) { r.tau[v] = 0.0; r.P[v] = __ldg(a.src_S + (size_t)r.src * NB + v) / npix0; }
                        STK(top + lane) = r;
                    }
                    top += n;
                    break;
                }
                // (3) nothing to do: wait for donations or for the end
                if (!registered_hungry) { if (lane == 0) atomicAdd(&sc->hungry, 1); registered_hungry = true; }
                int stop = 0;
                if (lane == 0) {
                    const long long inflight = ld_volatile_s64(&sc->in_flight);
                    if (inflight == 0 || ld_volatile_s32(&sc->error) != 0) stop = 1;
                    else {
                        const unsigned long long now = globaltimer_ns();
                        if (t_idle0 == 0 || inflight != last_seen) { t_idle0 = now; last_seen = inflight; }
                        else if (now - t_idle0 > 20000000000ull) { atomicCAS(&sc->error, 0, ARC_DEV_WATCHDOG); stop = 1; }
                    }
                }
                stop = __shfl_sync(0xffffffffu, stop, 0);
                if (stop) { quit = true; break; }
                __nanosleep(backoff);
                if (backoff < 2048) backoff *= 2;
            }
            if (registered_hungry && !quit) { if (lane == 0) atomicSub(&sc->hungry, 1); registered_hungry = false; }
            if (quit) break;
            __syncwarp();
        }

        // ------------------------------------------------------------------ pop a batch: lane = (family, child)
        const int nfam = (int)min((unsigned)ARC_BATCH_FAM, top - bot);
        top -= nfam;
        const int myfam = lane >> 2;
        bool active = myfam < nfam;
        uint32_t src = 0, pix = 0; int level = 0;
        double tau[NB], P[NB];
        const double INF = __longlong_as_double(0x7ff0000000000000ll);
        double tx = INF, ty = INF, tz = INF, r = 0, r_end = 0;
        [[maybe_unused]] double rthin = INF;   // FLAG_THIN: smallest radius at which this lane's ray stopped being optically thin
        unsigned ijk = 0;                      // cell coordinates, 10 bits each (N <= 1024)
        int cell = 0;                          // N <= 1024: N^3 <= 2^30
        int end = -1;
        unsigned long long h = 0; unsigned int seq = 0;
        if (active && a.blocked != nullptr) {                 // anisotropic emission: a blocked root ray does not exist
            const Rec *rp = &STK(top + myfam);
            if (rp->pad != 0) {                               // (a root above level l0 - thin start - is blocked with its level-l0 ancestor)
                const uint32_t p0 = (4u * rp->fam + (uint32_t)(lane & 3)) >> (2 * ((int)rp->level - a.l0));
                if (a.blocked[(size_t)rp->src * ((size_t)12 << (2 * a.l0)) + p0]) active = false;
            }
        }
        if (active) {
            const Rec *rp = &STK(top + myfam);
            src = rp->src; level = (int)rp->level; pix = 4u * rp->fam + (uint32_t)(lane & 3);
            ARC_CHECK(sc, src < (uint32_t)a.nsrc && level >= 0 && level < ARC_MAX_LEVEL && level <= a.Lmax && (unsigned long long)pix < (12ull << (2 * level)));
#pragma unroll
            for (int v = 0; v < NB; ++v) { tau[v] = rp->tau[v]; P[v] = rp->P[v]; }
            double dirx, diry, dirz;
            arc_pix2vec_dev(level, pix, dirx, diry, dirz);
            const double gx = __ldg(a.src_g + 3 * src), gy = __ldg(a.src_g + 3 * src + 1), gz = __ldg(a.src_g + 3 * src + 2);
            // the ray's constants live in shared memory (read back by this thread only: no barrier needed); the
            // loop fetches just the crossed axis' pair, which keeps 12 registers free for a third resident block
            // (stores and loads of s_geo are volatile asm: kept in program order among themselves)
#define GEO_ST(row, val) asm volatile("st.shared.f64 [%0+%1], %2;" ::"r"(geo_ad), "n"((row) * ARC_TRACE_THREADS * 8), "d"(val))
            GEO_ST(0, gx); GEO_ST(1, gy); GEO_ST(2, gz); GEO_ST(3, dirx); GEO_ST(4, diry); GEO_ST(5, dirz);
            // split radii: exact power-of-two scalings of csplit (O2)
            r = rp->pad != 0 ? (a.Rstart != nullptr ? __ldg(a.Rstart + src) : 0.0) : scalbn(a.csplit, level - 1);
            r_end = (level >= a.Lmax) ? INF : scalbn(a.csplit, level);
            // a5: starting cell (O3 step 2)
            const double x0 = arc_add(gx, arc_mul(r, dirx)), y0 = arc_add(gy, arc_mul(r, diry)), z0 = arc_add(gz, arc_mul(r, dirz));
            double fx = floor(x0), fy = floor(y0), fz = floor(z0);
            if (x0 == fx && dirx < 0.0) fx -= 1.0;
            if (y0 == fy && diry < 0.0) fy -= 1.0;
            if (z0 == fz && dirz < 0.0) fz -= 1.0;
            const double dN = (double)N;
            const bool inside = fx >= 0.0 && fx < dN && fy >= 0.0 && fy < dN && fz >= 0.0 && fz < dN;
            if (FLAGS & FLAG_DIGEST) h = mix64(((unsigned long long)src << 40) | ((unsigned long long)level << 32) | pix);
            atomicAdd(&s_rays[level], 1u);
            if (!inside) {
                end = ARC_END_ESCAPED; active = false;          // (P goes to the escape tally after the loop)
            } else {
                const int ix = (int)fx, iy = (int)fy, iz = (int)fz;
                ijk = (unsigned)ix | ((unsigned)iy << 10) | ((unsigned)iz << 20);
                cell = (iz * N + iy) * N + ix;
                if (dirx != 0.0) { tx = __ddiv_rn(arc_sub((double)(ix + (dirx > 0.0)), gx), dirx); GEO_ST(6, __ddiv_rn(1.0, dirx)); }
                if (diry != 0.0) { ty = __ddiv_rn(arc_sub((double)(iy + (diry > 0.0)), gy), diry); GEO_ST(7, __ddiv_rn(1.0, diry)); }
                if (dirz != 0.0) { tz = __ddiv_rn(arc_sub((double)(iz + (dirz > 0.0)), gz), dirz); GEO_ST(8, __ddiv_rn(1.0, dirz)); }
            }
        }

        // ------------------------------------------------------------------ a6/a7: the segment loop
        // One warp iteration = one (ray, cell) segment per active lane.  Everything that is per axis is selected once
        // (the crossed axis), the advance costs one IEEE division, the next cell's opacities are requested before this
        // segment's attenuation arithmetic, and the state advance is unconditional (a lane that just ended is inactive).
        unsigned int nseg_b = 0, nred_b = 0;     // (nseg_b also is this ray's segment count: one ray per lane and batch)
        // Geometric correction on the transposed route (GEOM_PIPE): the deposit runs ONE iteration late.  83 % of the shares
        // that Eq. 3 hands to the adjacent cell go to the ray's own next or previous cell (measured on the oracle's ray
        // logs, DESIGN.md 6.2 step 7): a share for the NEXT cell is carried in registers into the next segment's record, a
        // share for the PREVIOUS cell is added to that cell's record while it still waits in the staging area, and only
        // lateral shares need REDs of their own.  pcell = cell of the record waiting in my staging column.
        constexpr bool GEOM_PIPE = ((FLAGS & FLAG_GEOM) != 0) && DEP == DEP_T;
        [[maybe_unused]] double carry[NB];       // the share the last segment handed on (Eq. 3), until it has found its record
        [[maybe_unused]] int pcell = -1 - lane;
        [[maybe_unused]] bool have_carry = false; // ... it goes into this lane's next record
        [[maybe_unused]] int entry = -1;          // code (2 axis + [direction > 0]) of the crossing that led into the current cell; -1: first segment
        if constexpr (GEOM_PIPE) {
#pragma unroll
            for (int v = 0; v < NB; ++v) carry[v] = 0.0;
        }
        // DEP_T, stage 1: every lane writes its NB values into its column of the staging planes
        auto stage_store = [&](double (&val)[NB]) {
#pragma unroll
            for (int v = 0; v < NB; ++v) asm volatile("st.shared.f64 [%0], %1;" ::"r"(dep_wr + (unsigned)(v * DEP_PLANE)), "d"(val[v]) : "memory");
        };
        // DEP_T, stage 2: in pass k = 0..3 the 4 lanes of quad q send the record of ray 4q + k, lane (q, b) issues bin b (and
        // b + 4): the quad's REDs of one instruction fall in one 32-byte sector and leave the SM as one request - 2.5x the
        // RED rate of one lane walking through the record.  `key` = the cell of the record in my column (negative: none).
        auto stage_flush = [&](const int key) {
            ARC_CHECK(sc, key < a.NN * N);
            if constexpr (DEP == DEP_T) ARC_CHECK(sc, dep_wr + (unsigned)((NB - 1) * DEP_PLANE) + 8u <= (unsigned)__cvta_generic_to_shared(s_dep) + (unsigned)sizeof(s_dep)
                                                   && dep_rd + (unsigned)(((NB - 1) / 4 * 4) * DEP_PLANE) + 32u <= (unsigned)__cvta_generic_to_shared(s_dep) + (unsigned)sizeof(s_dep) + 3u * DEP_PLANE);
            // the quad's 4 rays are siblings (or 4 neighbouring root pixels) less than a cell apart: rays of the quad that
            // sit in the same cell are summed first (pure ALU work: the cells and values are in registers anyway), so a
            // cell gets one record per quad and iteration
            int cq[4];
            double vq[(NB + 3) / 4][4];
            // lane and bin from the (live) staging address instead of %tid (an S2R per iteration otherwise)
            const unsigned ln = (dep_wr >> 3) & 31u, bq = ln & 3u;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                cq[k] = __shfl_sync(0xffffffffu, key, (ln & ~3u) + k);
#pragma unroll
                for (int b0 = 0; b0 < NB; b0 += 4) {
                    vq[b0 / 4][k] = 0.0;
                    if (b0 + 4 <= NB || b0 + bq < NB)
                        asm volatile("ld.shared.f64 %0, [%1];" : "=d"(vq[b0 / 4][k]) : "r"(dep_rd + (unsigned)(b0 * DEP_PLANE + k * 8)) : "memory");
                }
            }
            // sums first (all lanes, no branches), then four predicated REDs
            bool first[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                first[k] = cq[k] >= 0;                           // not merged into an earlier ray of the quad
#pragma unroll
                for (int j = 0; j < k; ++j) first[k] = first[k] && (cq[j] != cq[k]);
#pragma unroll
                for (int j = k + 1; j < 4; ++j) {
                    const bool same = cq[j] == cq[k];
#pragma unroll
                    for (int b0 = 0; b0 < NB; b0 += 4) vq[b0 / 4][k] += same ? vq[b0 / 4][j] : 0.0;
                }
            }
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                // record index in 32 bits where it fits (N <= 1024: cells < 2^30): one LEA + one wide multiply-add
                double *Ac = (NBP <= 4) ? a.A + ((unsigned)cq[k] * (unsigned)NBP + bq) : a.A + (long long)cq[k] * NBP + bq;
#pragma unroll
                for (int b0 = 0; b0 < NB; b0 += 4)
                    arc_red_add_if(Ac + b0, vq[b0 / 4][k], first[k] && (b0 + 4 <= NB || b0 + bq < NB));
                if ((FLAGS & FLAG_DIGEST) && first[k] && bq == 0) ++nred_b;      // (statistic: digest builds only)
            }
        };
        KVec<KT, NB> kcur;
        ARC_CHECK(sc, (unsigned)cell < (unsigned)(a.NN * N));
        kcur.load(kappa, cell);                 // (cell 0 for lanes without a ray: harmless)
        for (;;) {
          if (!__any_sync(0xffffffffu, active)) break;
          double av[NB];
          int dcell = -1 - lane;                 // deposit key; lanes without a segment keep a unique negative one
          [[maybe_unused]] double avn[NB];       // FLAG_GEOM: what Eq. 3 hands to the adjacent cell ...
          [[maybe_unused]] int ncell = -1 - lane;  // ... and that cell (same convention as dcell)
          [[maybe_unused]] int cls = 0;          // GEOM_PIPE: where that share goes: 0 nowhere, 1 my previous cell, 2 my next cell, 3 a lateral cell
          [[maybe_unused]] int lat_code = 0;     // ... and the face it crosses (2 axis + upper)
          if (active) {
            // a6: first face crossed; ties go to x, then y (reading G9)
            int ax = 0; double tmin = tx;
            if (ty < tmin) { tmin = ty; ax = 1; }
            if (tz < tmin) { tmin = tz; ax = 2; }
            const bool split = (r_end <= tmin);
            const double r_out = split ? r_end : tmin;
            double ds = arc_sub(r_out, r);
            if (__double2hiint(ds) < 0) ds = 0.0;                          // max(ds, 0) (C4); ds is never NaN
            const double dl = arc_mul(ds, a.dx);
            double g_ax, d_ax, y_ax;
            {
                const unsigned ad = geo_ad + (unsigned)ax * (ARC_TRACE_THREADS * 8u);
                asm volatile("ld.shared.f64 %0, [%1];" : "=d"(g_ax) : "r"(ad));
                asm volatile("ld.shared.f64 %0, [%1+%2];" : "=d"(d_ax) : "r"(ad), "n"(3 * ARC_TRACE_THREADS * 8));
                asm volatile("ld.shared.f64 %0, [%1+%2];" : "=d"(y_ax) : "r"(ad), "n"(6 * ARC_TRACE_THREADS * 8));
            }
            const int pos = (__double2hiint(d_ax) >= 0) ? 1 : 0;          // d_ax > 0 (it is never zero on the crossed axis)
            const int st = 2 * pos - 1;
            const int sh = 10 * ax;
            const int inext = (int)((ijk >> sh) & 1023u) + st;
            const bool out = (unsigned)inext >= (unsigned)N;
            int stride = a.NN;
            if (ax == 1) stride = N;
            if (ax == 0) stride = 1;
            const int cell_next = cell + st * stride;
            const bool go = !(split || out);
            ARC_CHECK(sc, (unsigned)cell < (unsigned)(a.NN * N) && (!go || (unsigned)cell_next < (unsigned)(a.NN * N)) && ax >= 0 && ax <= 2);
            ARC_CHECK(sc, cell == (int)(((ijk >> 20) & 1023u) * (unsigned)N + ((ijk >> 10) & 1023u)) * N + (int)(ijk & 1023u));
            const double t_new = arc_div_by_recip(arc_sub((double)(inext + pos), g_ax), d_ax, y_ax);   // == IEEE division (C3)
            // a7: optical depth (fp64, decides: contract C4) and the deposit of Eq. 1
            bool depleted = true;
            if constexpr (sizeof(KT) == 4) {
                // fp32-field mode (tolerance 1e-3): the attenuation FACTOR is evaluated in fp32, two bins per packed
                // instruction (FMUL2 / FFMA2); everything that carries or decides stays fp64.  Thin segment (x < 1/64):
                // absorbed = P ome with ome = x (1 - x/2 + x^2/6 - x^3/24) (truncation < 5e-10), kept = P - absorbed;
                // otherwise kept = P E with E = 2^(-x log2 e) on the SFU, absorbed = P - kept (relative error of the
                // absorbed part <= 64 x 2 ulp = 1.5e-5).  Either way absorbed + kept = P to fp64 rounding.
                const float dlf = (float)dl;
                float x[NBE], om[NBE], y[NBE];
#pragma unroll
                for (int v = 0; v < NBE; v += 2) {
                    const unsigned long long xx = arc_mul2(arc_pack2(kcur.k[v], kcur.k[v + 1 < NB ? v + 1 : v]), arc_pack2(dlf, dlf));
                    unsigned long long pp = arc_fma2(arc_pack2(-1.0f / 24.0f, -1.0f / 24.0f), xx, arc_pack2(1.0f / 6.0f, 1.0f / 6.0f));
                    pp = arc_fma2(pp, xx, arc_pack2(-0.5f, -0.5f));
                    pp = arc_fma2(pp, xx, arc_pack2(1.0f, 1.0f));
                    pp = arc_mul2(pp, xx);
                    const unsigned long long yy = arc_mul2(xx, arc_pack2(-1.4426950408889634f, -1.4426950408889634f));
                    arc_unpack2(xx, x[v], x[v + 1]); arc_unpack2(pp, om[v], om[v + 1]); arc_unpack2(yy, y[v], y[v + 1]);
                }
                [[maybe_unused]] const double tau0_prev = tau[0];
#pragma unroll
                for (int v = 0; v < NB; ++v) {
                    tau[v] = arc_add(tau[v], arc_mul(kcur.get(v), dl));
                    depleted = depleted && (tau[v] >= a.tau_term);       // min_nu tau_nu >= tau_term
                }
                if constexpr ((FLAGS & FLAG_THIN) != 0) {                // (ii) of PAPER.md:120: tau reaches thin_tau in this segment,
                    if (tau0_prev < a.thin_tau && tau[0] >= a.thin_tau) rthin = fmin(rthin, r);     // which starts at radius r
                }
                // last use of kcur is above: the NEXT cell's opacities (always a valid cell: no divergence) go straight into
                // it and have the rest of this iteration, the deposit stage and the next march to arrive
                kcur.load(kappa, go ? cell_next : cell);
#pragma unroll
                for (int v = 0; v < NB; ++v) {
                    const bool thin = x[v] < 0.015625f;
                    const float f = thin ? om[v] : arc_ex2(y[v]);
                    const double q = P[v] * (double)f;
                    const double rest = P[v] - q;
                    av[v] = thin ? q : rest;
                    P[v] = thin ? rest : q;
                }
            } else {
                double dtau[NB];
                [[maybe_unused]] const double tau0_prev = tau[0];
#pragma unroll
                for (int v = 0; v < NB; ++v) {
                    dtau[v] = arc_mul(kcur.get(v), dl);
                    tau[v] = arc_add(tau[v], dtau[v]);
                    depleted = depleted && (tau[v] >= a.tau_term);
                }
                if constexpr ((FLAGS & FLAG_THIN) != 0) {
                    if (tau0_prev < a.thin_tau && tau[0] >= a.thin_tau) rthin = fmin(rthin, r);
                }
                kcur.load(kappa, go ? cell_next : cell);       // (as above)
#pragma unroll
                for (int v = 0; v < NB; ++v) {
                    double E, ome;
                    arc_attenuate(dtau[v], E, ome);             // e^-dtau and 1 - e^-dtau
                    av[v] = P[v] * ome;                         // absorbed = P (1 - e^-dtau)
                    P[v] = P[v] * E;                            // photon conserving: the ray keeps P e^-dtau
                }
            }
            if constexpr ((FLAGS & FLAG_GEOM) != 0) {
                // Geometric correction (readings G25-G29).  Which face is nearest decides where photons
                // go, so that part is contract arithmetic (explicit round-to-nearest operations in the oracle's order):
                // midpoint m_a = g_a + r_mid d_a, u_a = m_a - i_a, faces in the order x-, x+, y-, y+, z-, z+, first
                // minimum wins (taken per axis first - lower face unless the upper one is strictly nearer - then across the
                // axes, x before y before z: the same face as the oracle's scan); D_edge = max(min, 0);
                // L_pix = r_mid (cpix 2^-l); correction applies if 2 D_edge < L_pix.  The ray's own tau and P are not touched.
                const double rmid = arc_mul(0.5, arc_add(r, r_out));
                // cpix 2^-level: an exact power-of-two scaling, done on the exponent field (cpix ~ 1.02, level <= 14)
                const double Lpix = arc_mul(rmid, __hiloint2double(__double2hiint(a.cpix) - (level << 20), __double2loint(a.cpix)));
                double Dax[3]; int up[3];
#pragma unroll
                for (int ax3 = 0; ax3 < 3; ++ax3) {
                    double g3, d3;
                    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(g3) : "r"(geo_ad + (unsigned)(ax3 * ARC_TRACE_THREADS * 8)));
                    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(d3) : "r"(geo_ad + (unsigned)((3 + ax3) * ARC_TRACE_THREADS * 8)));
                    const double u = arc_sub(arc_add(g3, arc_mul(rmid, d3)), (double)((ijk >> (10 * ax3)) & 1023u));
                    const double hi = arc_sub(1.0, u);
                    up[ax3] = hi < u;
                    Dax[ax3] = up[ax3] ? hi : u;
                }
                double D = Dax[0]; int fcode = up[0];                       // face code = 2 axis + (upper face)
                if (Dax[1] < D) { D = Dax[1]; fcode = 2 + up[1]; }
                if (Dax[2] < D) { D = Dax[2]; fcode = 4 + up[2]; }
                if (__double2hiint(D) < 0) D = 0.0;                         // (rounding can put the midpoint a hair outside)
                bool corr = arc_mul(2.0, D) < Lpix;
                // f_c = 1/2 + D_edge / L_pix (Eq. 2) only weighs the deposit - it decides nothing - so the quotient need not be the
                // IEEE one; but it must be good to fp64: what goes to the neighbour is (1 - f_c) x absorbed, and f_c comes
                // arbitrarily close to 1 (an fp32 quotient put that share 3e-5 off in a few cells of a 4000-case sweep).
                // Hardware reciprocal seed + two Newton steps: ulp-level, 7 instructions against the ~17 of the division.
                double rL;
                asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(rL) : "d"(Lpix));
                rL = fma(fma(-Lpix, rL, 1.0), rL, rL);
                rL = fma(fma(-Lpix, rL, 1.0), rL, rL);
                double fc = 0.5 + fmin(D * rL, 0.5);                            // (the quotient is < 1/2 where it is used; NaN for L_pix = 0 -> 1/2, unused)
                if (a.geom == ARC_GEOM_FC2) fc = fc * fc;
                const int nax = fcode >> 1;
                const int jn = (int)((ijk >> (10 * nax)) & 1023u) + ((fcode & 1) ? 1 : -1);
                const bool nb_in = (unsigned)jn < (unsigned)N;
                // secondary correction with the neighbour outside the box: the cell keeps everything (G29)
                if (a.geom == ARC_GEOM_FC_SECONDARY && !nb_in) corr = false;
                if (!corr) fc = 1.0;                                        // (x 1.0 is exact: the deposit stays what it was)
                const bool move = corr && (a.geom == ARC_GEOM_FC_SECONDARY);
                if constexpr (GEOM_PIPE) {
                    // where the share goes: my previous cell lies across the face I entered through, my next cell across the face
                    // this segment ends on (if the ray goes on); anything else is a lateral cell
                    if (move) cls = (entry >= 0 && fcode == (entry ^ 1)) ? 1 : ((go && !depleted && fcode == 2 * ax + pos) ? 2 : 3);
                    lat_code = fcode;
                    // this cell's record = its own (corrected) absorption + what the previous segment handed forward; the share
                    // this segment hands on (Eq. 3) waits in `carry`
#pragma unroll
                    for (int v = 0; v < NB; ++v) {
                        double in = fc * av[v];
                        const double off = av[v] - in;
                        arc_add_if(in, carry[v], have_carry);
                        av[v] = in;
                        carry[v] = off;
                    }
                    have_carry = (cls == 2);
                    entry = 2 * ax + pos;                                   // (the face the next segment enters through)
                } else {
                    ncell = -1 - lane;
                    const int nstride = nax == 0 ? 1 : (nax == 1 ? N : a.NN);
                    if (move) ncell = cell + ((fcode & 1) ? nstride : -nstride);
#pragma unroll
                    for (int v = 0; v < NB; ++v) {
                        const double in = fc * av[v];
                        avn[v] = av[v] - in;                                  // (read only where ncell >= 0)
                        av[v] = in;
                    }
                }
            }
            dcell = cell;
            ++nseg_b;
            if (FLAGS & FLAG_DIGEST) h = mix64(h ^ (unsigned long long)cell);
            if (FLAGS & FLAG_LOG) {
                const unsigned long long e = atomicAdd(&sc->log_n, 1ull);
                if (e < a.log_cap) {
                    a.log_key[e] = ((unsigned long long)src << 40) | ((unsigned long long)level << 32) | pix;
                    a.log_seq[e] = seq; a.log_cell[e] = cell;
                }
                ++seq;
            }
            if (depleted || !go || nseg_b > a.max_seg) {
                active = false;
                if (depleted) {
                    end = ARC_END_DEPLETED;
#pragma unroll
                    for (int v = 0; v < NB; ++v) av[v] += P[v];     // reading G7: the remainder stays in this cell
                } else if (split) end = ARC_END_SPLIT;
                else {
                    if (!out) atomicCAS(&sc->error, 0, ARC_DEV_RAY_RUNAWAY);
                    end = ARC_END_ESCAPED;                      // what the ray still carries, P, leaves the box (a9): tallied after the loop
                }
            }
            // unconditional advance
            r = r_out; cell = cell_next;
            ijk += (unsigned)st << sh;
            tx = (ax == 0) ? t_new : tx;
            ty = (ax == 1) ? t_new : ty;
            tz = (ax == 2) ? t_new : tz;
          }
          // a7: deposit - the whole warp, converged
          auto deposit = [&](const int dcell, double (&av)[NB]) {
          if constexpr (DEP == DEP_AGG) {
              // segmented sum over the lanes that share a cell, by pointer jumping along each group's lane list:
              // after ceil(log2(group size)) rounds the first lane of a group holds the group's sum
              const unsigned peers = __match_any_sync(0xffffffffu, dcell);
              const int leader = __ffs(peers) - 1;
              int nxt = __ffs(peers & ~((2u << lane) - 1u)) - 1;          // next lane of my group, -1 at the tail
              while (__any_sync(0xffffffffu, nxt >= 0)) {
                  const int from = nxt >= 0 ? nxt : lane;
#pragma unroll
                  for (int v = 0; v < NB; ++v) {
                      const double o = __shfl_sync(0xffffffffu, av[v], from);
                      if (nxt >= 0) av[v] += o;
                  }
                  nxt = __shfl_sync(0xffffffffu, nxt, from);              // (a tail lane reads its own -1)
              }
              const bool head = (lane == leader);
              if (head && dcell >= 0) {
                  ARC_CHECK(sc, dcell < a.NN * N);
                  double *Ac = a.A + (long long)dcell * NBP;
#pragma unroll
                  for (int v = 0; v < NB; ++v) arc_red_add(Ac + v, av[v]);
                  ++nred_b;
              }
          } else if constexpr (DEP == DEP_T) {
              stage_store(av);
              __syncwarp();
              stage_flush(dcell);
              __syncwarp();                       // rows are rewritten in the next iteration
          } else {
              if (dcell >= 0) {
                  ARC_CHECK(sc, dcell < a.NN * N);
                  double *Ac = a.A + (long long)dcell * NBP;
#pragma unroll
                  for (int v = 0; v < NB; ++v) arc_red_add(Ac + v, av[v]);   // a7: REDG.E.ADD.F64 ("atomically")
                  ++nred_b;
              }
          }
          };
          if constexpr (GEOM_PIPE) {
              // the record in my staging column is that of my PREVIOUS segment (cell pcell): a share for that cell joins it there
              // (own column: no other lane writes it, and the quad read it before the last __syncwarp)
              if (cls == 1) {
#pragma unroll
                  for (int v = 0; v < NB; ++v) {
                      double x;
                      asm volatile("ld.shared.f64 %0, [%1];" : "=d"(x) : "r"(dep_wr + (unsigned)(v * DEP_PLANE)) : "memory");
                      x += carry[v];
                      asm volatile("st.shared.f64 [%0], %1;" ::"r"(dep_wr + (unsigned)(v * DEP_PLANE)), "d"(x) : "memory");
                  }
              }
              if (cls == 3) {                     // a lateral cell: REDs of its own (one lane, NB doubles of one record)
                  const int lax = lat_code >> 1, lstride = lax == 0 ? 1 : (lax == 1 ? N : a.NN);
                  ARC_CHECK(sc, (unsigned)(dcell + ((lat_code & 1) ? lstride : -lstride)) < (unsigned)(a.NN * N));
                  double *An = a.A + (long long)(dcell + ((lat_code & 1) ? lstride : -lstride)) * NBP;
#pragma unroll
                  for (int v = 0; v < NB; ++v) arc_red_add(An + v, carry[v]);
                  ++nred_b;
              }
              __syncwarp();
              stage_flush(pcell);                 // the records of the previous iteration, complete now
              __syncwarp();
              stage_store(av);                    // this iteration's records wait for the next one
              pcell = dcell;
          } else {
              deposit(dcell, av);
              if constexpr ((FLAGS & FLAG_GEOM) != 0) {
                  if (__any_sync(0xffffffffu, ncell >= 0)) deposit(ncell, avn);        // Eq. 3: the adjacent cells' share
              }
          }
        }
        if constexpr (GEOM_PIPE) {
            // the records of the last iteration are still waiting
            __syncwarp();
            stage_flush(pcell);
            __syncwarp();
        }
        nseg += nseg_b; nred += nred_b;
        __syncwarp();

        // ------------------------------------------------------------------ a8/a9: bookkeeping, push children
        if constexpr ((FLAGS & FLAG_THIN) != 0) {
            // a ray that left the box or was depleted while still thin: thin up to where it ended (r is its final radius)
            if ((end == ARC_END_ESCAPED || end == ARC_END_DEPLETED) && tau[0] < a.thin_tau) rthin = fmin(rthin, r);
            if (rthin < INF) {
                const unsigned long long bits = (unsigned long long)__double_as_longlong(rthin);    // radii >= 0: bits order as values
                if (bits < ld_volatile_u64(a.Rnext + src)) atomicMin(a.Rnext + src, bits);           // (values only decrease: a stale read is safe)
            }
        }
        {
            // a9 tallies, once per batch and warp: rays by end reason (ballots), photons that left the box (warp sum of P
            // over the lanes whose ray escaped; P is untouched once a ray has ended)
            const unsigned e0 = __ballot_sync(0xffffffffu, end == 0), e1 = __ballot_sync(0xffffffffu, end == 1), e2 = __ballot_sync(0xffffffffu, end == 2);
            if (lane < 3) { const unsigned n = __popc(lane == 0 ? e0 : (lane == 1 ? e1 : e2)); if (n) atomicAdd(&s_ends[lane], n); }
            if (e2) {
#pragma unroll
                for (int v = 0; v < NB; ++v) {
                    double e = (end == ARC_END_ESCAPED) ? P[v] : 0.0;
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
                    if (lane == 0) atomicAdd(&s_esc[v], e);
                }
            }
        }
        if (end >= 0) {
            if (FLAGS & FLAG_DIGEST) { h = mix64(h ^ (0xE0ull + (unsigned long long)end)); digest += h; }
            if (FLAGS & FLAG_LOG) {
                const unsigned long long e = atomicAdd(&sc->log_n, 1ull);
                if (e < a.log_cap) {
                    a.log_key[e] = ((unsigned long long)src << 40) | ((unsigned long long)level << 32) | pix;
                    a.log_seq[e] = seq; a.log_cell[e] = -1 - end;
                }
            }
        }
        const bool do_split = (end == ARC_END_SPLIT);
        if (do_split) atomicAdd(&s_splits[level], 1u);
        const unsigned ballot = __ballot_sync(0xffffffffu, do_split);
        const int npush = __popc(ballot);
        if (top - bot + npush > ARC_STACK_CAP) {
            if (lane == 0) atomicCAS(&sc->error, 0, ARC_DEV_STACK_OVERFLOW);
            quit = true;
        } else {
            if (do_split) {
                const int rank = __popc(ballot & ((1u << lane) - 1u));
                ARC_CHECK(sc, level + 1 <= a.Lmax && top + rank - bot < ARC_STACK_CAP);
                Rec rec;
                rec.src = src; rec.fam = pix; rec.level = (uint32_t)(level + 1); rec.pad = 0;
#pragma unroll
                for (int v = 0; v < NB; ++v) { rec.tau[v] = tau[v]; rec.P[v] = 0.25 * P[v]; }     // each child: a quarter
                STK(top + rank) = rec;
            }
            top += npush;
            delta += (long long)npush - nfam;
        }
        __syncwarp();

        // ------------------------------------------------------------------ donate the shallow end of the ring if someone is idle
        int hungry = 0, err = 0;
        if (lane == 0) { hungry = ld_volatile_s32(&sc->hungry); err = ld_volatile_s32(&sc->error); }
        hungry = __shfl_sync(0xffffffffu, hungry, 0);
        err = __shfl_sync(0xffffffffu, err, 0);
        if (err) quit = true;
        const unsigned nd_max = min(top - bot > (unsigned)ARC_DONATE_KEEP ? top - bot - (unsigned)ARC_DONATE_KEEP : 0u, 32u);   // keep the next batch, give the rest
        if (!quit && hungry > 0 && nd_max > 0) {
            int nd = (int)nd_max;
            unsigned long long ticket = 0;
            if (lane == 0) {
                // donate only while the pool is short of what the idle warps can take; the level test is
                // approximate (plain loads), the ring is sized so that every warp overshooting at once still fits
                const unsigned long long t = ld_volatile_u64(&sc->q_tail), hq = ld_volatile_u64(&sc->q_head);
                const unsigned long long level_now = t > hq ? t - hq : 0ull;
                if (level_now >= (unsigned long long)min(hungry * ARC_POOL_PER_HUNGRY, ARC_QUEUE_LOW)) nd = 0;
                else {
                    // flush first: donated families must be covered by the global counter before they are visible
                    if (delta != 0) atomicAdd((unsigned long long *)&sc->in_flight, (unsigned long long)delta);
                    ticket = atomicAdd(&sc->q_tail, (unsigned long long)nd);
                    atomicMax(&sc->q_high, ticket + nd - hq);
                }
            }
            nd = __shfl_sync(0xffffffffu, nd, 0);
            ticket = __shfl_sync(0xffffffffu, ticket, 0);
            if (nd > 0) {
                delta = 0;
                if (lane < nd) {
                    const unsigned long long tk = ticket + lane;
                    const unsigned slot = (unsigned)(tk % ARC_QUEUE_CAP);
                    ARC_CHECK(sc, bot + lane < top);
                    while (ld_volatile_u64(&a.qseq[slot]) != tk) __nanosleep(32);    // previous lap's reader finished
                    const int4 *s4 = reinterpret_cast<const int4 *>(&STK(bot + lane));
                    int4 *d4 = reinterpret_cast<int4 *>(&queue[slot]);
#pragma unroll
                    for (int w = 0; w < (int)(sizeof(Rec) / 16); ++w) __stcg(d4 + w, s4[w]);
                    __threadfence();
                    *(volatile unsigned long long *)&a.qseq[slot] = tk + 1;            // publish
                }
                __syncwarp();
                if (lane == 0) atomicAdd((unsigned long long *)&sc->q_count, (unsigned long long)nd);
            }
            bot += nd;
            __syncwarp();
        }
    }

    // ---------------------------------------------------------------------- flush statistics
    if (registered_hungry && lane == 0) atomicSub(&sc->hungry, 1);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        nseg += __shfl_xor_sync(0xffffffffu, nseg, o);
        nred += __shfl_xor_sync(0xffffffffu, nred, o);
        digest += __shfl_xor_sync(0xffffffffu, digest, o);
    }
    if (lane == 0) {
        atomicAdd(&a.stats->segments, nseg);
        atomicAdd(&a.stats->segments_total, nseg);
        atomicAdd(&a.stats->deposit_records, nred);
        if (FLAGS & FLAG_DIGEST) atomicAdd(&a.stats->digest, digest);
    }
    __syncthreads();
    if (threadIdx.x < ARC_MAX_LEVEL) {
        if (s_splits[threadIdx.x]) atomicAdd(&a.stats->splits[threadIdx.x], (unsigned long long)s_splits[threadIdx.x]);
        if (s_rays[threadIdx.x]) { atomicAdd(&a.stats->rays_level[threadIdx.x], (unsigned long long)s_rays[threadIdx.x]); atomicAdd(&a.stats->rays, (unsigned long long)s_rays[threadIdx.x]); }
    }
    if (threadIdx.x < 3 && s_ends[threadIdx.x]) atomicAdd(&a.stats->ends[threadIdx.x], (unsigned long long)s_ends[threadIdx.x]);
    if (threadIdx.x < NB && s_esc[threadIdx.x] != 0.0) atomicAdd(&a.stats->escaped[threadIdx.x], s_esc[threadIdx.x]);
}

template <int NB, typename KT, int DEP>
cudaError_t launch_dep(const TraceArgs &a, bool log, int grid, cudaStream_t s)
{
    if (a.flags & FLAG_THIN) {                   // AUTO deposit route, no geometric correction, no ray log (arc_set_params / arc_trace_debug check)
        if constexpr (DEP == (NB >= 3 ? DEP_T : DEP_AGG)) {
            if (log || (a.flags & FLAG_GEOM)) return cudaErrorInvalidValue;
            if (a.flags & FLAG_DIGEST) arc_trace_kernel<NB, KT, FLAG_THIN | FLAG_DIGEST, DEP><<<grid, ARC_TRACE_THREADS, 0, s>>>(a);
            else arc_trace_kernel<NB, KT, FLAG_THIN, DEP><<<grid, ARC_TRACE_THREADS, 0, s>>>(a);
            return cudaGetLastError();
        } else return cudaErrorInvalidValue;
    }
    if (a.flags & FLAG_GEOM) {                   // built for the AUTO deposit route of this bin count only (arc_set_params checks)
        if constexpr (DEP == (NB >= 3 ? DEP_T : DEP_AGG)) {
            if (log) arc_trace_kernel<NB, KT, FLAG_GEOM | FLAG_LOG | FLAG_DIGEST, DEP><<<grid, ARC_TRACE_THREADS, 0, s>>>(a);
            else if (a.flags & FLAG_DIGEST) arc_trace_kernel<NB, KT, FLAG_GEOM | FLAG_DIGEST, DEP><<<grid, ARC_TRACE_THREADS, 0, s>>>(a);
            else arc_trace_kernel<NB, KT, FLAG_GEOM, DEP><<<grid, ARC_TRACE_THREADS, 0, s>>>(a);
            return cudaGetLastError();
        } else return cudaErrorInvalidValue;
    }
    if (log) arc_trace_kernel<NB, KT, FLAG_LOG | FLAG_DIGEST, DEP><<<grid, ARC_TRACE_THREADS, 0, s>>>(a);
    else if (a.flags & FLAG_DIGEST) arc_trace_kernel<NB, KT, FLAG_DIGEST, DEP><<<grid, ARC_TRACE_THREADS, 0, s>>>(a);
    else arc_trace_kernel<NB, KT, 0, DEP><<<grid, ARC_TRACE_THREADS, 0, s>>>(a);
    return cudaGetLastError();
}

template <int NB, typename KT>
cudaError_t launch_nb(const TraceArgs &a, bool log, int dep, int grid, cudaStream_t s)
{
    switch (dep) {
        case DEP_AGG: return launch_dep<NB, KT, DEP_AGG>(a, log, grid, s);
        case DEP_T: return launch_dep<NB, KT, DEP_T>(a, log, grid, s);
        default: return launch_dep<NB, KT, DEP_RED>(a, log, grid, s);
    }
}

template <int NB, typename KT, int DEP>
int occ_dep(int flags)
{
    int nblk = 0;
    cudaError_t e;
    if (flags & FLAG_THIN) {
        if constexpr (DEP == (NB >= 3 ? DEP_T : DEP_AGG)) {
            if (flags & FLAG_DIGEST) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nblk, arc_trace_kernel<NB, KT, FLAG_THIN | FLAG_DIGEST, DEP>, ARC_TRACE_THREADS, 0);
            else e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nblk, arc_trace_kernel<NB, KT, FLAG_THIN, DEP>, ARC_TRACE_THREADS, 0);
        } else e = cudaErrorInvalidValue;
        if (e != cudaSuccess) { cudaGetLastError(); return 1; }
        return nblk < 1 ? 1 : nblk;
    }
    if (flags & FLAG_GEOM) {
        if constexpr (DEP == (NB >= 3 ? DEP_T : DEP_AGG)) {
            if (flags & FLAG_LOG) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nblk, arc_trace_kernel<NB, KT, FLAG_GEOM | FLAG_LOG | FLAG_DIGEST, DEP>, ARC_TRACE_THREADS, 0);
            else if (flags & FLAG_DIGEST) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nblk, arc_trace_kernel<NB, KT, FLAG_GEOM | FLAG_DIGEST, DEP>, ARC_TRACE_THREADS, 0);
            else e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nblk, arc_trace_kernel<NB, KT, FLAG_GEOM, DEP>, ARC_TRACE_THREADS, 0);
        } else e = cudaErrorInvalidValue;
        if (e != cudaSuccess) { cudaGetLastError(); return 1; }
        return nblk < 1 ? 1 : nblk;
    }
    if (flags & FLAG_LOG) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nblk, arc_trace_kernel<NB, KT, FLAG_LOG | FLAG_DIGEST, DEP>, ARC_TRACE_THREADS, 0);
    else if (flags & FLAG_DIGEST) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nblk, arc_trace_kernel<NB, KT, FLAG_DIGEST, DEP>, ARC_TRACE_THREADS, 0);
    else e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nblk, arc_trace_kernel<NB, KT, 0, DEP>, ARC_TRACE_THREADS, 0);
    if (e != cudaSuccess) { cudaGetLastError(); return 1; }
    return nblk < 1 ? 1 : nblk;
}

template <int NB, typename KT>
int occ_nb(int dep, int flags)
{
    return dep == DEP_AGG ? occ_dep<NB, KT, DEP_AGG>(flags) : dep == DEP_T ? occ_dep<NB, KT, DEP_T>(flags) : occ_dep<NB, KT, DEP_RED>(flags);
}

}  // namespace

// One translation unit per (opacity dtype, half of the bin range): ARC_INST_KT, ARC_INST_NB0 (1 or 5), ARC_INST_TAG
#define ARC_CAT2(a, b) a##b
#define ARC_CAT(a, b) ARC_CAT2(a, b)

cudaError_t ARC_CAT(arc_trace_launch_, ARC_INST_TAG)(const TraceArgs &a, bool log, int dep, int grid, cudaStream_t s)
{
    switch (a.nb - ARC_INST_NB0) {
        case 0: return launch_nb<ARC_INST_NB0 + 0, ARC_INST_KT>(a, log, dep, grid, s);
        case 1: return launch_nb<ARC_INST_NB0 + 1, ARC_INST_KT>(a, log, dep, grid, s);
        case 2: return launch_nb<ARC_INST_NB0 + 2, ARC_INST_KT>(a, log, dep, grid, s);
        case 3: return launch_nb<ARC_INST_NB0 + 3, ARC_INST_KT>(a, log, dep, grid, s);
    }
    return cudaErrorInvalidValue;
}

int ARC_CAT(arc_trace_occ_, ARC_INST_TAG)(int nb, int dep, int flags)
{
    switch (nb - ARC_INST_NB0) {
        case 0: return occ_nb<ARC_INST_NB0 + 0, ARC_INST_KT>(dep, flags);
        case 1: return occ_nb<ARC_INST_NB0 + 1, ARC_INST_KT>(dep, flags);
        case 2: return occ_nb<ARC_INST_NB0 + 2, ARC_INST_KT>(dep, flags);
        case 3: return occ_nb<ARC_INST_NB0 + 3, ARC_INST_KT>(dep, flags);
    }
    return 1;
}
