// arc_trace.cu -- the persistent ray-tracing kernel.
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
//    warps donate the shallow half of their stack (biggest subtrees) through a bounded MPMC ticket queue.
//  * Deterministic arithmetic (contract C0-C5): every operation that decides a cell, an axis, a split or a
//    termination is an explicit IEEE round-to-nearest intrinsic (no FMA contraction), typed from DESIGN.md.
#include "arc_internal.cuh"
#include "arc_healpix.cuh"

#define FLAG_LOG 1
#define FLAG_DIGEST 2

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

// ---------------------------------------------------------------------------------------------------
template <int NB, typename KT, int FLAGS>
__global__ void __launch_bounds__(ARC_TRACE_THREADS, 2) arc_trace_kernel(const TraceArgs a)
{
    typedef FamRec<NB> Rec;
    const int lane = threadIdx.x & 31;
    const int gwarp = blockIdx.x * ARC_WARPS_PER_BLOCK + (threadIdx.x >> 5);
    Rec *const stack = reinterpret_cast<Rec *>(a.stacks) + (size_t)gwarp * ARC_STACK_CAP;
    Rec *const queue = reinterpret_cast<Rec *>(a.queue);
    SchedState *const sc = a.sched;
    const KT *const kappa = reinterpret_cast<const KT *>(a.kappa);
    const int N = a.N;

    __shared__ unsigned long long s_splits[ARC_MAX_LEVEL], s_rays[ARC_MAX_LEVEL], s_ends[3];
    __shared__ double s_esc[ARC_MAX_BINS];
    if (threadIdx.x < ARC_MAX_LEVEL) { s_splits[threadIdx.x] = 0; s_rays[threadIdx.x] = 0; }
    if (threadIdx.x < 3) s_ends[threadIdx.x] = 0;
    if (threadIdx.x < ARC_MAX_BINS) s_esc[threadIdx.x] = 0.0;
    __syncthreads();

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
                        const int hungry_now = max(ld_volatile_s32(&sc->hungry), 1);
                        const long long want = max(1ll, min((long long)ARC_BATCH_FAM, avail / hungry_now));
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
                        r.src = (uint32_t)(s / a.fam_per_src); r.fam = (uint32_t)(s % a.fam_per_src);
                        r.level = (uint32_t)a.l0; r.pad = 0;
#pragma unroll
                        for (int v = 0; v < NB; ++v) r.tau[v] = 0.0;
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
        double gx = 0, gy = 0, gz = 0, dirx = 0, diry = 0, dirz = 0, tx = 0, ty = 0, tz = 0, r = 0, r_end = 0;
        int ix = 0, iy = 0, iz = 0, sx = 0, sy = 0, sz = 0;
        int cell = 0;                          // N <= 1024: N^3 <= 2^30
        int end = -1;
        unsigned long long h = 0; unsigned int seq = 0;
        if (active) {
            const Rec *rp = &STK(top + myfam);
            src = rp->src; level = (int)rp->level; pix = 4u * rp->fam + (uint32_t)(lane & 3);
#pragma unroll
            for (int v = 0; v < NB; ++v) tau[v] = rp->tau[v];
            arc_pix2vec_dev(level, pix, dirx, diry, dirz);
            gx = __ldg(a.src_g + 3 * src); gy = __ldg(a.src_g + 3 * src + 1); gz = __ldg(a.src_g + 3 * src + 2);
            const double npix = (double)(12ull << (2 * level));
#pragma unroll
            for (int v = 0; v < NB; ++v) P[v] = (__ldg(a.src_S + (size_t)src * NB + v) / npix) * exp(-tau[v]);
            // split radii: exact power-of-two scalings of csplit (O2)
            r = (level == a.l0) ? 0.0 : scalbn(a.csplit, level - 1);
            r_end = (level >= a.Lmax) ? __longlong_as_double(0x7ff0000000000000ll) : scalbn(a.csplit, level);
            // a5: starting cell (O3 step 2)
            const double x0 = arc_add(gx, arc_mul(r, dirx)), y0 = arc_add(gy, arc_mul(r, diry)), z0 = arc_add(gz, arc_mul(r, dirz));
            double fx = floor(x0), fy = floor(y0), fz = floor(z0);
            if (x0 == fx && dirx < 0.0) fx -= 1.0;
            if (y0 == fy && diry < 0.0) fy -= 1.0;
            if (z0 == fz && dirz < 0.0) fz -= 1.0;
            const double dN = (double)N;
            const bool inside = fx >= 0.0 && fx < dN && fy >= 0.0 && fy < dN && fz >= 0.0 && fz < dN;
            if (FLAGS & FLAG_DIGEST) h = mix64(((unsigned long long)src << 40) | ((unsigned long long)level << 32) | pix);
            atomicAdd(&s_rays[level], 1ull);
            if (!inside) {
#pragma unroll
                for (int v = 0; v < NB; ++v) atomicAdd(&s_esc[v], P[v]);
                end = ARC_END_ESCAPED; active = false;
            } else {
                ix = (int)fx; iy = (int)fy; iz = (int)fz;
                cell = (iz * N + iy) * N + ix;
                sx = dirx > 0.0 ? 1 : (dirx < 0.0 ? -1 : 0);
                sy = diry > 0.0 ? 1 : (diry < 0.0 ? -1 : 0);
                sz = dirz > 0.0 ? 1 : (dirz < 0.0 ? -1 : 0);
                const double INF = __longlong_as_double(0x7ff0000000000000ll);
                tx = sx ? __ddiv_rn(arc_sub((double)(ix + (sx > 0)), gx), dirx) : INF;
                ty = sy ? __ddiv_rn(arc_sub((double)(iy + (sy > 0)), gy), diry) : INF;
                tz = sz ? __ddiv_rn(arc_sub((double)(iz + (sz > 0)), gz), dirz) : INF;
            }
        }

        // ------------------------------------------------------------------ a6/a7: the segment loop
        // One iteration = one (ray, cell) segment.  The axis advance is branch-free (one IEEE division per
        // segment, whichever axis is crossed) and the next cell's opacities are requested BEFORE this segment's
        // attenuation arithmetic, so the gather latency hides behind it.
        const unsigned int max_seg = 3u * (unsigned)N + 8u;
        unsigned int nray_seg = 0;
        KVec<KT, NB> kcur;
        if (active) kcur.load(kappa, cell);
        while (active) {
            int ax = 0; double tmin = tx;
            if (ty < tmin) { tmin = ty; ax = 1; }
            if (tz < tmin) { tmin = tz; ax = 2; }
            const bool split = (r_end <= tmin);
            const double r_out = split ? r_end : tmin;
            const double dl = arc_mul(fmax(arc_sub(r_out, r), 0.0), a.dx);
            // a6: where the ray goes next (used only if it neither splits nor ends here)
            const int st = ax == 0 ? sx : (ax == 1 ? sy : sz);
            const int inext = (ax == 0 ? ix : (ax == 1 ? iy : iz)) + st;
            const bool out = (unsigned)inext >= (unsigned)N;
            const int stride = ax == 0 ? 1 : (ax == 1 ? N : N * N);
            const int cell_next = cell + st * stride;
            KVec<KT, NB> knext;
            if (!split && !out) knext.load(kappa, cell_next);
            const double g_ax = ax == 0 ? gx : (ax == 1 ? gy : gz);
            const double d_ax = ax == 0 ? dirx : (ax == 1 ? diry : dirz);
            const double t_new = __ddiv_rn(arc_sub((double)(inext + (st > 0)), g_ax), d_ax);
            // a7: optical depth and deposit (Eq. 1)
            double av[NB];
            double taumin = __longlong_as_double(0x7ff0000000000000ll);
#pragma unroll
            for (int v = 0; v < NB; ++v) {
                const double dtau = arc_mul(kcur.get(v), dl);
                tau[v] = arc_add(tau[v], dtau);                 // decides termination: IEEE, no FMA (C4)
                taumin = fmin(taumin, tau[v]);
                double E, ome;
                arc_attenuate(dtau, E, ome);                    // e^-dtau and 1 - e^-dtau
                av[v] = P[v] * ome;                             // absorbed = P (1 - e^-dtau)
                P[v] = P[v] * E;                                // photon conserving: the ray keeps P e^-dtau
            }
            const bool depleted = (taumin >= a.tau_term);
            double *Ac = a.A + (long long)cell * NB;
#pragma unroll
            for (int v = 0; v < NB; ++v) {
                if (depleted) av[v] += P[v];                    // reading G7: the remainder stays in this cell
                arc_red_add(Ac + v, av[v]);                     // a7: RED.ADD.F64 ("atomically")
            }
            ++nseg; ++nray_seg;
            if (FLAGS & FLAG_DIGEST) h = mix64(h ^ (unsigned long long)cell);
            if (FLAGS & FLAG_LOG) {
                const unsigned long long e = atomicAdd(&sc->log_n, 1ull);
                if (e < a.log_cap) {
                    a.log_key[e] = ((unsigned long long)src << 40) | ((unsigned long long)level << 32) | pix;
                    a.log_seq[e] = seq; a.log_cell[e] = cell;
                }
                ++seq;
            }
            if (depleted) { end = ARC_END_DEPLETED; active = false; }
            else if (split) { end = ARC_END_SPLIT; active = false; }
            else if (out) {
#pragma unroll
                for (int v = 0; v < NB; ++v) atomicAdd(&s_esc[v], P[v]);
                end = ARC_END_ESCAPED; active = false;
            } else if (nray_seg > max_seg) { atomicCAS(&sc->error, 0, ARC_DEV_RAY_RUNAWAY); end = ARC_END_ESCAPED; active = false; }
            else {
                r = r_out; cell = cell_next; kcur = knext;
                if (ax == 0) { ix = inext; tx = t_new; } else if (ax == 1) { iy = inext; ty = t_new; } else { iz = inext; tz = t_new; }
            }
        }
        __syncwarp();

        // ------------------------------------------------------------------ a8/a9: bookkeeping, push children
        if (end >= 0) {
            atomicAdd(&s_ends[end], 1ull);
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
        if (do_split) atomicAdd(&s_splits[level], 1ull);
        const unsigned ballot = __ballot_sync(0xffffffffu, do_split);
        const int npush = __popc(ballot);
        if (top - bot + npush > ARC_STACK_CAP) {
            if (lane == 0) atomicCAS(&sc->error, 0, ARC_DEV_STACK_OVERFLOW);
            quit = true;
        } else {
            if (do_split) {
                const int rank = __popc(ballot & ((1u << lane) - 1u));
                Rec rec;
                rec.src = src; rec.fam = pix; rec.level = (uint32_t)(level + 1); rec.pad = 0;
#pragma unroll
                for (int v = 0; v < NB; ++v) rec.tau[v] = tau[v];
                STK(top + rank) = rec;
            }
            top += npush;
            delta += (long long)npush - nfam;
        }
        __syncwarp();

        // ------------------------------------------------------------------ donate the shallow half if someone is idle
        int hungry = 0, err = 0;
        if (lane == 0) { hungry = ld_volatile_s32(&sc->hungry); err = ld_volatile_s32(&sc->error); }
        hungry = __shfl_sync(0xffffffffu, hungry, 0);
        err = __shfl_sync(0xffffffffu, err, 0);
        if (err) quit = true;
        if (!quit && hungry > 0 && top - bot >= 2) {
            int nd = (int)min((top - bot) / 2, 32u);
            unsigned long long ticket = 0;
            if (lane == 0) {
                // donate only while the pool is short of what the idle warps can take; the level test is
                // approximate (plain loads), the ring is sized so that every warp overshooting at once still fits
                const unsigned long long t = ld_volatile_u64(&sc->q_tail), hq = ld_volatile_u64(&sc->q_head);
                const unsigned long long level_now = t > hq ? t - hq : 0ull;
                if (level_now >= (unsigned long long)min(hungry * 4, ARC_QUEUE_LOW)) nd = 0;
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
        digest += __shfl_xor_sync(0xffffffffu, digest, o);
    }
    if (lane == 0) {
        atomicAdd(&a.stats->segments, nseg);
        if (FLAGS & FLAG_DIGEST) atomicAdd(&a.stats->digest, digest);
    }
    __syncthreads();
    if (threadIdx.x < ARC_MAX_LEVEL) {
        if (s_splits[threadIdx.x]) atomicAdd(&a.stats->splits[threadIdx.x], s_splits[threadIdx.x]);
        if (s_rays[threadIdx.x]) { atomicAdd(&a.stats->rays_level[threadIdx.x], s_rays[threadIdx.x]); atomicAdd(&a.stats->rays, s_rays[threadIdx.x]); }
    }
    if (threadIdx.x < 3 && s_ends[threadIdx.x]) atomicAdd(&a.stats->ends[threadIdx.x], s_ends[threadIdx.x]);
    if (threadIdx.x < NB && s_esc[threadIdx.x] != 0.0) atomicAdd(&a.stats->escaped[threadIdx.x], s_esc[threadIdx.x]);
}

template <int NB, typename KT>
cudaError_t launch_nb(const TraceArgs &a, int flags, int grid, cudaStream_t s)
{
    switch (flags) {
        case 0: arc_trace_kernel<NB, KT, 0><<<grid, ARC_TRACE_THREADS, 0, s>>>(a); break;
        case FLAG_DIGEST: arc_trace_kernel<NB, KT, FLAG_DIGEST><<<grid, ARC_TRACE_THREADS, 0, s>>>(a); break;
        default: arc_trace_kernel<NB, KT, FLAG_LOG | FLAG_DIGEST><<<grid, ARC_TRACE_THREADS, 0, s>>>(a); break;
    }
    return cudaGetLastError();
}

template <typename KT>
cudaError_t launch_kt(const TraceArgs &a, int flags, int grid, cudaStream_t s)
{
    switch (a.nb) {
        case 1: return launch_nb<1, KT>(a, flags, grid, s);
        case 2: return launch_nb<2, KT>(a, flags, grid, s);
        case 3: return launch_nb<3, KT>(a, flags, grid, s);
        case 4: return launch_nb<4, KT>(a, flags, grid, s);
        case 5: return launch_nb<5, KT>(a, flags, grid, s);
        case 6: return launch_nb<6, KT>(a, flags, grid, s);
        case 7: return launch_nb<7, KT>(a, flags, grid, s);
        case 8: return launch_nb<8, KT>(a, flags, grid, s);
    }
    return cudaErrorInvalidValue;
}

template <int NB, typename KT>
int occ_nb()
{
    int nblk = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nblk, arc_trace_kernel<NB, KT, 0>, ARC_TRACE_THREADS, 0) != cudaSuccess) return 1;
    return nblk < 1 ? 1 : nblk;
}

// scheduler reset before each trace: all root families are "in flight", queue empty, slot i expects ticket i
__global__ void arc_sched_reset_kernel(SchedState *sc, DevStats *st, unsigned long long *qseq, unsigned long long seed_total)
{
    const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < ARC_QUEUE_CAP) qseq[i] = i;
    if (i == 0) {
        sc->in_flight = (long long)seed_total; sc->seed_next = 0; sc->q_head = 0; sc->q_tail = 0;
        sc->hungry = 0; sc->error = ARC_DEV_OK; sc->q_high = 0; sc->log_n = 0; sc->q_count = 0;
        st->segments = 0; st->rays = 0; st->digest = 0;
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

int arc_trace_occupancy_grid(arc_ctx *c, int nb)
{
    int per_sm = 1;
    const bool f32 = (c->dtype == ARC_F32);
    switch (nb) {
        case 1: per_sm = f32 ? occ_nb<1, float>() : occ_nb<1, double>(); break;
        case 2: per_sm = f32 ? occ_nb<2, float>() : occ_nb<2, double>(); break;
        case 3: per_sm = f32 ? occ_nb<3, float>() : occ_nb<3, double>(); break;
        case 4: per_sm = f32 ? occ_nb<4, float>() : occ_nb<4, double>(); break;
        case 5: per_sm = f32 ? occ_nb<5, float>() : occ_nb<5, double>(); break;
        case 6: per_sm = f32 ? occ_nb<6, float>() : occ_nb<6, double>(); break;
        case 7: per_sm = f32 ? occ_nb<7, float>() : occ_nb<7, double>(); break;
        default: per_sm = f32 ? occ_nb<8, float>() : occ_nb<8, double>(); break;
    }
    return c->n_sm * per_sm;
}

cudaError_t arc_launch_trace(arc_ctx *c, const TraceArgs &a, bool log, int *grid_out)
{
    const int flags = log ? (FLAG_LOG | FLAG_DIGEST) : (c->p.digest ? FLAG_DIGEST : 0);
    const int grid = c->trace_grid;
    if (grid_out) *grid_out = grid;
    return (c->dtype == ARC_F32) ? launch_kt<float>(a, flags, grid, c->stream) : launch_kt<double>(a, flags, grid, c->stream);
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
