// arc_trace.cu -- host side of the persistent tracer: deposit-mode choice, dispatch to the instantiation units
// (arc_trace_inst_*.cu), scheduler reset and the exposed pix2vec kernel.  The kernel itself is arc_trace_kernel.cuh.
#include "arc_internal.cuh"
#include "arc_healpix.cuh"
#include "arc_divide.cuh"

#define DECL_INST(tag)                                                                                        \
    cudaError_t arc_trace_launch_##tag(const TraceArgs &a, bool log, int dep, int grid, cudaStream_t s);      \
    int arc_trace_occ_##tag(int nb, int dep, int flags);
DECL_INST(f32_lo) DECL_INST(f32_hi) DECL_INST(f64_lo) DECL_INST(f64_hi)

namespace {

// Full reset of the donation queue: slot i expects ticket i, tickets start at 0.  Needed before the first trace and after
// a trace that aborted; a trace that ends cleanly leaves the queue drained and consistent (every published ticket was
// consumed, slot s then expects the next ticket that maps to it), so tickets simply keep counting from one trace to the
// next and the 2 MB of slot words are not rewritten per trace.  The per-trace words are reset by arc_opacity_kernel.
__global__ void arc_queue_reset_kernel(SchedState *sc, unsigned long long *qseq)
{
    const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < ARC_QUEUE_CAP) qseq[i] = i;
    if (i == 0) { sc->q_head = 0; sc->q_tail = 0; sc->q_count = 0; sc->hungry = 0; }
}

__global__ void arc_pix2vec_kernel(const int32_t *level, const uint32_t *pix, int n, double *out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double x, y, z;
    arc_pix2vec_dev(level[i], pix[i], x, y, z);
    out[3 * i] = x; out[3 * i + 1] = y; out[3 * i + 2] = z;
}

// ---- arc_selftest_division: arc_div_by_recip against __ddiv_rn on device-generated operands -------------------------
__device__ __forceinline__ unsigned long long st_mix(unsigned long long x)      // splitmix64 finaliser (counter-based generator)
{
    x ^= x >> 30; x *= 0xbf58476d1ce4e5b9ull;
    x ^= x >> 27; x *= 0x94d049bb133111ebull;
    x ^= x >> 31;
    return x;
}

// pair number k -> (a, d) in the ranges the march produces (include/arc.h): a = i - g, d = a direction component
__device__ __forceinline__ void st_pair(unsigned long long seed, unsigned long long k, double &a, double &d)
{
    const unsigned long long r0 = st_mix(seed + 0x9e3779b97f4a7c15ull * (2 * k + 1)), r1 = st_mix(r0 ^ 0xd1b54a32d192ed03ull), r2 = st_mix(r1 + k);
    // direction component: exponent uniform in [-40, 0], 52 random mantissa bits; special shapes by the low bits of r2
    const int e = -(int)(r0 % 41u);
    unsigned long long man = r1 >> 12;
    switch (r2 & 7u) {
        case 0: man = 0x000fffffffffffffull - (r1 & 3u); break;          // just below the next power of two
        case 1: man = r1 & 3u; break;                                    // at / just above a power of two
        case 2: man &= 0x000ffff000000000ull; break;                     // short mantissa
        default: break;
    }
    d = __longlong_as_double((long long)(((unsigned long long)(1023 + e) << 52) | man));
    if (d > 1.0) d = 1.0;
    if (r2 & 8u) d = -d;
    // source coordinate in [0, 1024): 53-bit uniform, or snapped to a grid of 1, 1/2, 2^-10 (sources on faces / centres)
    double g = (double)(r2 >> 11) * (1024.0 / 9007199254740992.0);
    switch ((r2 >> 4) & 7u) {
        case 0: g = floor(g); break;
        case 1: g = floor(g) + 0.5; break;
        case 2: g = floor(g * 1024.0) / 1024.0; break;
        default: break;
    }
    const int i = (int)((r0 >> 32) % 1026u);                             // cell face index 0 .. 1025
    a = __dsub_rn((double)i, g);
}

__global__ void __launch_bounds__(256) arc_selftest_division_kernel(unsigned long long n, unsigned long long seed, unsigned long long *bad)
{
    unsigned long long mine = 0;
    for (unsigned long long k = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; k < n; k += (unsigned long long)gridDim.x * blockDim.x) {
        double a, d;
        st_pair(seed, k, a, d);
        const double y = __ddiv_rn(1.0, d);
        const double q = arc_div_by_recip(a, d, y), ref = __ddiv_rn(a, d);
        if (__double_as_longlong(q) != __double_as_longlong(ref)) ++mine;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mine += __shfl_xor_sync(0xffffffffu, mine, o);
    if ((threadIdx.x & 31) == 0 && mine) atomicAdd(bad, mine);
}

}  // namespace

extern "C" int arc_selftest_division(uint64_t n_pairs, uint64_t seed, uint64_t *mismatches)
{
    if (!mismatches) return ARC_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return ARC_ECUDA; }
    unsigned long long *d_bad = nullptr, h = 0;
    cudaError_t e = cudaMalloc(&d_bad, sizeof(h));
    if (e == cudaSuccess) e = cudaMemset(d_bad, 0, sizeof(h));
    if (e == cudaSuccess && n_pairs > 0) {
        arc_selftest_division_kernel<<<148 * 8, 256>>>((unsigned long long)n_pairs, (unsigned long long)seed, d_bad);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpy(&h, d_bad, sizeof(h), cudaMemcpyDeviceToHost);
    cudaFree(d_bad);
    if (e != cudaSuccess) { cudaGetLastError(); return ARC_ECUDA; }
    *mismatches = h;
    return ARC_OK;
}

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
    ++c->launches;
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

cudaError_t arc_launch_queue_reset(arc_ctx *c)
{
    arc_queue_reset_kernel<<<ARC_QUEUE_CAP / 256, 256, 0, c->stream>>>(c->d_sched, c->d_qseq);
    ++c->launches;
    return cudaGetLastError();
}
