// arc_fields.cu -- per-cell streaming kernels around the tracer.
//   a1+a2 fused: zero the accumulators and build the opacity table
//           kappa_nu = (sigma_HI,nu n_HI + sigma_HeI,nu n_HeI) + sigma_HeII,nu n_HeII
//         evaluated in fp64 left to right and rounded to the field dtype (O4).
//   a10: finalise  Gamma_S = (1/V) sum_nu A_nu sigma_S,nu / kappa'_nu,  heat_S likewise with (E_nu - E_S)
//         (Eq. 1 with n_abs = n_SI; species share = opacity share, reading G8).
// SoA fields (5 arrays at the field dtype) are read fully coalesced, one cell per thread.
#include "arc_internal.cuh"

namespace {

__device__ __forceinline__ double n_helium(double nH, double Yp) { return nH * Yp / (4.0 * (1.0 - Yp)); }

template <typename FT>
__global__ void __launch_bounds__(256) arc_opacity_kernel(long long ncell, int nb, int nbp, double Yp, Spectrum sp,
                                                         const FT *__restrict__ nH, const FT *__restrict__ xHI,
                                                         const FT *__restrict__ xHeI, const FT *__restrict__ xHeII,
                                                         FT *__restrict__ kappa, double *__restrict__ A,
                                                         SchedState *sc, DevStats *st, double *absorbed, unsigned long long seed_total, int fault)
{
    // per-trace reset of the scheduler words and tallies (the tracer is the next kernel on the stream): all root families
    // are "in flight".  The error word is STICKY: what an earlier asynchronous trace left behind, and the host has not yet
    // seen and cleared (arc_check_device), stays - the tracer then does not run and every consumer kernel keeps skipping.
    // `fault` = arc_params.debug_fault (test hook).
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        sc->in_flight = (long long)seed_total; sc->seed_next = 0; sc->hungry = 0; sc->q_high = 0; sc->log_n = 0;
        if (sc->error == ARC_DEV_OK) sc->error = fault;
        st->segments = 0; st->rays = 0; st->digest = 0; st->deposit_records = 0;
        for (int l = 0; l < ARC_MAX_LEVEL; ++l) { st->splits[l] = 0; st->rays_level[l] = 0; }
        for (int e = 0; e < 3; ++e) st->ends[e] = 0;
        for (int v = 0; v < ARC_MAX_BINS; ++v) { st->escaped[v] = 0.0; absorbed[v] = 0.0; }
    }
    for (long long c = blockIdx.x * (long long)blockDim.x + threadIdx.x; c < ncell; c += (long long)gridDim.x * blockDim.x) {
        const double n = (double)nH[c];
        const double nHe = n_helium(n, Yp);
        const double nHI = __dmul_rn(n, (double)xHI[c]);
        const double nHeI = __dmul_rn(nHe, (double)xHeI[c]);
        const double nHeII = __dmul_rn(nHe, (double)xHeII[c]);
        for (int v = 0; v < nb; ++v) {
            const double k = __dadd_rn(__dadd_rn(__dmul_rn(sp.sig[0][v], nHI), __dmul_rn(sp.sig[1][v], nHeI)),
                                       __dmul_rn(sp.sig[2][v], nHeII));
            kappa[c * nb + v] = (FT)k;
        }
        for (int v = 0; v < nbp; ++v) A[c * nbp + v] = 0.0;
    }
}

template <typename FT>
__global__ void __launch_bounds__(256) arc_finalize_kernel(long long ncell, int nb, int nbp, double Yp, double V, Spectrum sp,
                                                          const FT *__restrict__ nH, const FT *__restrict__ xHI,
                                                          const FT *__restrict__ xHeI, const FT *__restrict__ xHeII,
                                                          const double *__restrict__ A, double *__restrict__ rates,
                                                          double *__restrict__ absorbed, const SchedState *__restrict__ sc)
{
    // async mode: a trace that aborted on the device (sticky error word, or families left in flight) has no valid
    // accumulators - leave the rates alone; the host reports the error at its next synchronising call
    if (sc->error != ARC_DEV_OK || sc->in_flight != 0) return;
    const double EV = 1.602176634e-12;
    const double ETH[3] = {13.598, 24.587, 54.418};
    double acc[ARC_MAX_BINS];
#pragma unroll
    for (int v = 0; v < ARC_MAX_BINS; ++v) acc[v] = 0.0;
    for (long long c = blockIdx.x * (long long)blockDim.x + threadIdx.x; c < ncell; c += (long long)gridDim.x * blockDim.x) {
        const double n = (double)nH[c];
        const double nHe = n_helium(n, Yp);
        const double ns[3] = {n * (double)xHI[c], nHe * (double)xHeI[c], nHe * (double)xHeII[c]};
        double G[3] = {0.0, 0.0, 0.0}, H[3] = {0.0, 0.0, 0.0};
#pragma unroll
        for (int v = 0; v < ARC_MAX_BINS; ++v) {
            if (v >= nb) break;
            const double Av = A[c * nbp + v];
            acc[v] += Av;
            const double kp = (sp.sig[0][v] * ns[0] + sp.sig[1][v] * ns[1]) + sp.sig[2][v] * ns[2];
            if (kp > 0.0) {
                const double w = Av / (V * kp);
#pragma unroll
                for (int S = 0; S < 3; ++S) {
                    const double ws = w * sp.sig[S][v];
                    G[S] += ws;
                    if (sp.E[v] > ETH[S]) H[S] += ws * ((sp.E[v] - ETH[S]) * EV);
                }
            }
        }
#pragma unroll
        for (int S = 0; S < 3; ++S) { rates[S * ncell + c] = G[S]; rates[(3 + S) * ncell + c] = H[S]; }
        rates[6 * ncell + c] = (H[0] * ns[0] + H[1] * ns[1]) + H[2] * ns[2];
    }
    // stats: absorbed_nu = sum over cells of A_nu (photon-conservation check)
    __shared__ double sm[ARC_MAX_BINS][8];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int v = 0; v < ARC_MAX_BINS; ++v) {
        double x = acc[v];
        for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
        if (lane == 0) sm[v][w] = x;
    }
    __syncthreads();
    if (threadIdx.x < nb) {
        double x = 0.0;
        for (int i = 0; i < 8; ++i) x += sm[threadIdx.x][i];
        atomicAdd(absorbed + threadIdx.x, x);
    }
}

}  // namespace

static int stream_grid(arc_ctx *c, long long n)
{
    long long b = (n + 255) / 256;
    const long long cap = (long long)c->n_sm * 16;      // grid-stride: a multiple of the SM count
    return (int)(b < cap ? b : cap);
}

cudaError_t arc_launch_opacity(arc_ctx *c, unsigned long long seed_total)
{
    const int g = stream_grid(c, c->ncell);
    if (c->dtype == ARC_F32)
        arc_opacity_kernel<float><<<g, 256, 0, c->stream>>>(c->ncell, c->spec.nb, arc_nbp(c->spec.nb), c->p.Yp, c->spec, (const float *)c->f[0],
                                                          (const float *)c->f[1], (const float *)c->f[2], (const float *)c->f[3],
                                                          (float *)c->d_kappa, c->d_A, c->d_sched, c->d_stats, c->d_absorbed, seed_total, c->p.debug_fault);
    else
        arc_opacity_kernel<double><<<g, 256, 0, c->stream>>>(c->ncell, c->spec.nb, arc_nbp(c->spec.nb), c->p.Yp, c->spec, (const double *)c->f[0],
                                                           (const double *)c->f[1], (const double *)c->f[2], (const double *)c->f[3],
                                                           (double *)c->d_kappa, c->d_A, c->d_sched, c->d_stats, c->d_absorbed, seed_total, c->p.debug_fault);
    ++c->launches;
    return cudaGetLastError();
}

// Optically thin inner region (PAPER.md:116-130 (iii); readings G33-G37): for every source with Rstart > 0, each cell
// whose centre lies within Rstart receives S_nu kappa_nu V / (4 pi r^2) absorbed photons/s (Eq. 1 for small tau with the
// dilution 4 pi r^2; r^2 not below (d/2)^2).  blockIdx.y = source, blockIdx.x/threadIdx.x = cell of the cube of side
// 2 ceil(maxR) + 1 around the source's cell.  Membership (d2 <= R^2) is contract arithmetic in the oracle's order.
template <typename FT>
__global__ void __launch_bounds__(256) arc_thin_region_kernel(int N, int nsrc, int nb, int nbp, int side, double dx, const double *__restrict__ src_g,
                                                             const double *__restrict__ Rstart, const double *__restrict__ Sopen,
                                                             const FT *__restrict__ kappa, double *__restrict__ A)
{
  for (int s = blockIdx.y; s < nsrc; s += gridDim.y) {
    const double R = Rstart[s];
    if (!(R > 0.0)) continue;
    const double gx = src_g[3 * s], gy = src_g[3 * s + 1], gz = src_g[3 * s + 2];
    const int h = side / 2;
    const int cx = (int)floor(gx), cy = (int)floor(gy), cz = (int)floor(gz);
    const double R2 = __dmul_rn(R, R);
    const double PI = 3.14159265358979323846;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < (long long)side * side * side; t += (long long)gridDim.x * blockDim.x) {
        const int ix = cx - h + (int)(t % side), iy = cy - h + (int)((t / side) % side), iz = cz - h + (int)(t / ((long long)side * side));
        if ((unsigned)ix >= (unsigned)N || (unsigned)iy >= (unsigned)N || (unsigned)iz >= (unsigned)N) continue;
        const double ex = __dsub_rn(__dadd_rn((double)ix, 0.5), gx), ey = __dsub_rn(__dadd_rn((double)iy, 0.5), gy), ez = __dsub_rn(__dadd_rn((double)iz, 0.5), gz);
        const double d2 = __dadd_rn(__dadd_rn(__dmul_rn(ex, ex), __dmul_rn(ey, ey)), __dmul_rn(ez, ez));
        if (!(d2 <= R2)) continue;
        const double r2 = d2 < 0.25 ? 0.25 : d2;
        const long long c = ((long long)iz * N + iy) * N + ix;
        for (int v = 0; v < nb; ++v) {
            const double a_v = Sopen[(size_t)s * nb + v] * ((double)kappa[c * nb + v] * dx) / (4.0 * PI * r2);
            atomicAdd(A + c * nbp + v, a_v);
        }
    }
  }
}

cudaError_t arc_launch_thin_region(arc_ctx *c, double maxR)
{
    int side = 2 * (int)ceil(maxR) + 3;
    if (side > 2 * c->N + 1) side = 2 * c->N + 1;
    const long long cells = (long long)side * side * side;
    long long gx = (cells + 255) / 256;
    if (gx > 1024) gx = 1024;
    const dim3 grid((unsigned)gx, (unsigned)(c->nsrc < 65535 ? c->nsrc : 65535));
    const int nb = c->spec.nb;
    if (c->dtype == ARC_F32)
        arc_thin_region_kernel<float><<<grid, 256, 0, c->stream>>>(c->N, c->nsrc, nb, arc_nbp(nb), side, c->dx, c->d_src_g, c->d_Rstart, c->d_Sopen,
                                                                  (const float *)c->d_kappa, c->d_A);
    else
        arc_thin_region_kernel<double><<<grid, 256, 0, c->stream>>>(c->N, c->nsrc, nb, arc_nbp(nb), side, c->dx, c->d_src_g, c->d_Rstart, c->d_Sopen,
                                                                   (const double *)c->d_kappa, c->d_A);
    ++c->launches;
    return cudaGetLastError();
}

cudaError_t arc_launch_finalize(arc_ctx *c)
{
    const int g = stream_grid(c, c->ncell);
    const double V = c->dx * c->dx * c->dx;
    if (c->dtype == ARC_F32)
        arc_finalize_kernel<float><<<g, 256, 0, c->stream>>>(c->ncell, c->spec.nb, arc_nbp(c->spec.nb), c->p.Yp, V, c->spec, (const float *)c->f[0],
                                                           (const float *)c->f[1], (const float *)c->f[2], (const float *)c->f[3],
                                                           c->d_A, c->d_rates, c->d_absorbed, c->d_sched);
    else
        arc_finalize_kernel<double><<<g, 256, 0, c->stream>>>(c->ncell, c->spec.nb, arc_nbp(c->spec.nb), c->p.Yp, V, c->spec, (const double *)c->f[0],
                                                            (const double *)c->f[1], (const double *)c->f[2], (const double *)c->f[3],
                                                            c->d_A, c->d_rates, c->d_absorbed, c->d_sched);
    ++c->launches;
    return cudaGetLastError();
}
