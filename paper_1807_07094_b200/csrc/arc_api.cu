// arc_api.cu -- the C ABI of include/arc.h: context, copies in and out, launch sequencing, error reporting.
// No arithmetic of the method lives here except the two host scalars the kernels take (source position in
// grid units g = pos/dx, and c = sqrt(3/(pi Phi)), O2/O3) - IEEE divide/sqrt, identical anywhere.
#include "arc_internal.cuh"
#include <cmath>
#include <cstring>
#include <new>
#include <vector>

static thread_local std::string g_create_err;

#define CK(call)                                                                                              \
    do {                                                                                                      \
        cudaError_t e_ = (call);                                                                              \
        if (e_ != cudaSuccess) {                                                                              \
            c->err = std::string(#call) + ": " + cudaGetErrorString(e_);                                      \
            return e_ == cudaErrorMemoryAllocation ? ARC_ENOMEM : ARC_ECUDA;                                  \
        }                                                                                                     \
    } while (0)

static int fail(arc_ctx *c, int code, const std::string &msg)
{
    if (c) c->err = msg; else g_create_err = msg;
    return code;
}

static size_t esize(const arc_ctx *c) { return c->dtype == ARC_F32 ? 4 : 8; }

extern "C" {

#ifdef ARC_CHECKED
const char *arc_version(void) { return "arc-b200 0.2 (sm_100a, checked build)"; }
#else
const char *arc_version(void) { return "arc-b200 0.2 (sm_100a)"; }
#endif

const char *arc_last_error(const arc_ctx *c) { return c ? c->err.c_str() : g_create_err.c_str(); }

void arc_default_params(arc_params *p)
{
    std::memset(p, 0, sizeof(*p));
    p->l0 = 1; p->Lmax = 13; p->Phi = 3.0; p->tau_term = 30.0; p->Yp = 0.0;
    p->isothermal = 1; p->caseB = 1; p->coll_ion = 0; p->max_subcycles = 4096;
    p->eps_sub = 0.1; p->x_floor = 1e-12; p->digest = 0; p->async = 0; p->trace_blocks = 0; p->deposit = ARC_DEPOSIT_AUTO; p->geom_corr = ARC_GEOM_NONE; p->debug_fault = 0; p->thin_tau = 0.0;
}

int arc_create_grid(arc_ctx **out, int N, double box_cm, int dtype)
{
    if (!out) return fail(nullptr, ARC_EINVAL, "arc_create_grid: out is NULL");
    *out = nullptr;
    if (N < 1 || N > 1024) return fail(nullptr, ARC_EINVAL, "arc_create_grid: N must be in [1, 1024]");
    if (!(box_cm > 0.0) || !std::isfinite(box_cm)) return fail(nullptr, ARC_EINVAL, "arc_create_grid: box_cm must be positive");
    if (dtype != ARC_F32 && dtype != ARC_F64) return fail(nullptr, ARC_EINVAL, "arc_create_grid: dtype must be ARC_F32 or ARC_F64");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(nullptr, ARC_ECUDA, "arc_create_grid: no CUDA device (there is no CPU fallback)");
    }
    arc_ctx *c = new (std::nothrow) arc_ctx();
    if (!c) return fail(nullptr, ARC_ENOMEM, "arc_create_grid: host allocation failed");
    c->N = N; c->dtype = dtype; c->box_cm = box_cm; c->dx = box_cm / (double)N;
    c->ncell = (int64_t)N * N * N;
    arc_default_params(&c->p);
    std::memset(&c->spec, 0, sizeof(c->spec));
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceProp prop;
    cudaError_t e = cudaGetDeviceProperties(&prop, dev);
    if (e == cudaSuccess && prop.major < 10) {
        delete c;
        return fail(nullptr, ARC_ECUDA, "arc_create_grid: device is not sm_100 class (this library is built for sm_100a only)");
    }
    c->n_sm = (e == cudaSuccess) ? prop.multiProcessorCount : 148;
    for (int i = 0; i < 5 && e == cudaSuccess; ++i) e = cudaMalloc(&c->f[i], (size_t)c->ncell * esize(c));
    if (e == cudaSuccess) e = cudaMalloc(&c->d_rates, (size_t)c->ncell * 7 * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc(&c->d_sched, sizeof(SchedState));
    if (e == cudaSuccess) e = cudaMalloc(&c->d_stats, sizeof(DevStats));
    if (e == cudaSuccess) e = cudaMalloc(&c->d_absorbed, sizeof(double) * ARC_MAX_BINS);
    if (e == cudaSuccess) e = cudaMemset(c->d_stats, 0, sizeof(DevStats));
    if (e == cudaSuccess) e = cudaMemset(c->d_sched, 0, sizeof(SchedState));      // (the error word is sticky across resets)
    if (e == cudaSuccess) e = cudaMemset(c->d_absorbed, 0, sizeof(double) * ARC_MAX_BINS);
    for (int i = 0; i < 8 && e == cudaSuccess; ++i) e = cudaEventCreate(&c->ev[i]);
    if (e != cudaSuccess) {
        g_create_err = std::string("arc_create_grid: ") + cudaGetErrorString(e);
        const int code = (e == cudaErrorMemoryAllocation) ? ARC_ENOMEM : ARC_ECUDA;
        arc_destroy(c);
        cudaGetLastError();
        return code;
    }
    *out = c;
    return ARC_OK;
}

int arc_destroy(arc_ctx *c)
{
    if (!c) return ARC_OK;
    cudaStreamSynchronize(c->stream);
    for (int i = 0; i < 5; ++i) cudaFree(c->f[i]);
    cudaFree(c->d_rates); cudaFree(c->d_sched); cudaFree(c->d_stats); cudaFree(c->d_absorbed); cudaFree(c->d_dt); cudaFree(c->d_blocked);
    cudaFree(c->d_Rstart); cudaFree(c->d_Rnext); cudaFree(c->d_seed_prefix); cudaFree(c->d_src_level); cudaFree(c->d_Sopen);
    cudaFree(c->d_kappa); cudaFree(c->d_A); cudaFree(c->d_src_g); cudaFree(c->d_src_S);
    cudaFree(c->d_stacks); cudaFree(c->d_queue); cudaFree(c->d_qseq);
    for (int i = 0; i < 8; ++i) if (c->ev[i]) cudaEventDestroy(c->ev[i]);
    for (int i = 0; i < 2; ++i) if (c->ev_steps[i]) cudaEventDestroy(c->ev_steps[i]);
    if (c->step_exec) cudaGraphExecDestroy(c->step_exec);
    delete c;
    return ARC_OK;
}

int arc_set_params(arc_ctx *c, const arc_params *p)
{
    if (!c || !p) return fail(c, ARC_EINVAL, "arc_set_params: NULL argument");
    if (p->l0 < 0 || p->l0 > 10) return fail(c, ARC_EINVAL, "arc_set_params: l0 must be in [0, 10]");
    if (p->Lmax < p->l0 || p->Lmax > 14) return fail(c, ARC_EINVAL, "arc_set_params: Lmax must be in [l0, 14]");
    if (!(p->Phi > 0.0) || !std::isfinite(p->Phi)) return fail(c, ARC_EINVAL, "arc_set_params: Phi must be positive");
    if (!(p->tau_term > 0.0)) return fail(c, ARC_EINVAL, "arc_set_params: tau_term must be positive (or +inf)");
    if (!(p->Yp >= 0.0 && p->Yp < 1.0)) return fail(c, ARC_EINVAL, "arc_set_params: Yp must be in [0, 1)");
    if (p->max_subcycles < 1) return fail(c, ARC_EINVAL, "arc_set_params: max_subcycles must be >= 1");
    if (!(p->eps_sub > 0.0)) return fail(c, ARC_EINVAL, "arc_set_params: eps_sub must be positive");
    if (!(p->x_floor >= 0.0 && p->x_floor < 1.0)) return fail(c, ARC_EINVAL, "arc_set_params: x_floor must be in [0, 1)");
    if (p->trace_blocks < 0) return fail(c, ARC_EINVAL, "arc_set_params: trace_blocks must be >= 0");
    if (p->deposit < ARC_DEPOSIT_AUTO || p->deposit > ARC_DEPOSIT_QUAD) return fail(c, ARC_EINVAL, "arc_set_params: bad deposit mode");
    if (p->debug_fault < 0 || p->debug_fault > ARC_DEV_RAY_RUNAWAY) return fail(c, ARC_EINVAL, "arc_set_params: debug_fault must be 0 or a device error code (1..4)");
    if (p->geom_corr < ARC_GEOM_NONE || p->geom_corr > ARC_GEOM_FC2) return fail(c, ARC_EINVAL, "arc_set_params: bad geom_corr");
    if (!(p->thin_tau >= 0.0) || !std::isfinite(p->thin_tau)) return fail(c, ARC_EINVAL, "arc_set_params: thin_tau must be finite and >= 0");
    if (p->thin_tau > 0.0 && (p->geom_corr != ARC_GEOM_NONE || p->deposit != ARC_DEPOSIT_AUTO))
        return fail(c, ARC_EINVAL, "arc_set_params: the optically thin region is built for deposit = AUTO and geom_corr = NONE only");
    if (p->geom_corr != ARC_GEOM_NONE && p->deposit != ARC_DEPOSIT_AUTO)
        return fail(c, ARC_EINVAL, "arc_set_params: the geometric correction is built for deposit = ARC_DEPOSIT_AUTO only");
    c->p = *p;
    c->have_rates = false; c->have_accum = false; ++c->epoch;
    return ARC_OK;
}

int arc_set_stream(arc_ctx *c, void *cuda_stream)
{
    if (!c) return ARC_EINVAL;
    cudaStreamSynchronize(c->stream);
    c->stream = (cudaStream_t)cuda_stream; ++c->epoch;
    return ARC_OK;
}

int arc_set_fields(arc_ctx *c, const void *n_H, const void *x_HI, const void *x_HeI, const void *x_HeII, const void *T, int where)
{
    if (!c) return ARC_EINVAL;
    if (where != ARC_HOST && where != ARC_DEVICE) return fail(c, ARC_EINVAL, "arc_set_fields: bad `where`");
    const void *src[5] = {n_H, x_HI, x_HeI, x_HeII, T};
    for (int i = 0; i < 5; ++i)
        if (!src[i] && !c->have_fields) return fail(c, ARC_EINVAL, "arc_set_fields: all five fields are needed on the first call");
    const cudaMemcpyKind kind = (where == ARC_HOST) ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice;
    for (int i = 0; i < 5; ++i)
        if (src[i]) CK(cudaMemcpyAsync(c->f[i], src[i], (size_t)c->ncell * esize(c), kind, c->stream));
    if (where == ARC_HOST) CK(cudaStreamSynchronize(c->stream));     // the caller may reuse pageable buffers
    c->have_fields = true;
    c->have_rates = false; c->have_accum = false;
    return ARC_OK;
}

int arc_get_fields(arc_ctx *c, void *n_H, void *x_HI, void *x_HeI, void *x_HeII, void *T, int where)
{
    if (!c) return ARC_EINVAL;
    if (where != ARC_HOST && where != ARC_DEVICE) return fail(c, ARC_EINVAL, "arc_get_fields: bad `where`");
    if (!c->have_fields) return fail(c, ARC_ESTATE, "arc_get_fields: no fields set");
    void *dst[5] = {n_H, x_HI, x_HeI, x_HeII, T};
    const cudaMemcpyKind kind = (where == ARC_HOST) ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice;
    for (int i = 0; i < 5; ++i)
        if (dst[i]) CK(cudaMemcpyAsync(dst[i], c->f[i], (size_t)c->ncell * esize(c), kind, c->stream));
    if (where == ARC_HOST) { CK(cudaStreamSynchronize(c->stream)); if (c->unchecked) return arc_check_device(c); }
    return ARC_OK;
}

int arc_set_spectrum(arc_ctx *c, int nbins, const double *E_eV, const double *sig_HI, const double *sig_HeI, const double *sig_HeII)
{
    if (!c) return ARC_EINVAL;
    if (nbins < 1 || nbins > ARC_MAX_BINS) return fail(c, ARC_EINVAL, "arc_set_spectrum: nbins must be in [1, ARC_MAX_BINS]");
    if (!E_eV || !sig_HI || !sig_HeI || !sig_HeII) return fail(c, ARC_EINVAL, "arc_set_spectrum: NULL argument");
    for (int v = 0; v < nbins; ++v) {
        if (!(E_eV[v] > 0.0) || !(sig_HI[v] >= 0.0) || !(sig_HeI[v] >= 0.0) || !(sig_HeII[v] >= 0.0))
            return fail(c, ARC_EINVAL, "arc_set_spectrum: energies must be positive and cross-sections non-negative");
    }
    CK(cudaStreamSynchronize(c->stream));
    if (nbins != c->spec.nb || !c->d_kappa) {
        cudaFree(c->d_kappa); cudaFree(c->d_A); c->d_kappa = nullptr; c->d_A = nullptr;
        CK(cudaMalloc(&c->d_kappa, (size_t)c->ncell * nbins * esize(c)));
        CK(cudaMalloc(&c->d_A, (size_t)c->ncell * arc_nbp(nbins) * sizeof(double)));
        if (c->have_src && nbins != c->spec.nb) c->have_src = false;      // binfrac rows no longer match
    }
    std::memset(&c->spec, 0, sizeof(c->spec));
    c->spec.nb = nbins;
    for (int v = 0; v < nbins; ++v) {
        c->spec.E[v] = E_eV[v]; c->spec.sig[0][v] = sig_HI[v]; c->spec.sig[1][v] = sig_HeI[v]; c->spec.sig[2][v] = sig_HeII[v];
    }
    c->have_spec = true;
    c->have_rates = false; c->have_accum = false; ++c->epoch;
    return ARC_OK;
}

int arc_set_sources(arc_ctx *c, int nsrc, const double *pos_cm, const double *Ndot, const double *binfrac)
{
    if (!c) return ARC_EINVAL;
    if (!c->have_spec) return fail(c, ARC_ESTATE, "arc_set_sources: call arc_set_spectrum first");
    if (nsrc < 0 || nsrc > (1 << 24)) return fail(c, ARC_EINVAL, "arc_set_sources: nsrc must be in [0, 2^24]");
    if (nsrc > 0 && (!pos_cm || !Ndot || !binfrac)) return fail(c, ARC_EINVAL, "arc_set_sources: NULL argument");
    const int nb = c->spec.nb;
    std::vector<double> g((size_t)nsrc * 3), S((size_t)nsrc * nb);
    for (int v = 0; v < ARC_MAX_BINS; ++v) c->emitted[v] = 0.0;
    for (int s = 0; s < nsrc; ++s) {
        for (int a = 0; a < 3; ++a) {
            const double x = pos_cm[3 * s + a];
            if (!(x >= 0.0 && x < c->box_cm)) return fail(c, ARC_EINVAL, "arc_set_sources: source position outside [0, box)");
            const double gg = x / c->dx;                            // grid units
            if (!(gg < (double)c->N)) return fail(c, ARC_EINVAL, "arc_set_sources: source position rounds onto the upper box face (pos / (box / N) >= N): no cell");
            g[3 * (size_t)s + a] = gg;
        }
        if (!(Ndot[s] >= 0.0) || !std::isfinite(Ndot[s])) return fail(c, ARC_EINVAL, "arc_set_sources: Ndot must be finite and >= 0");
        for (int v = 0; v < nb; ++v) {
            const double f = binfrac[(size_t)s * nb + v];
            if (!(f >= 0.0) || !std::isfinite(f)) return fail(c, ARC_EINVAL, "arc_set_sources: binfrac must be finite and >= 0");
            S[(size_t)s * nb + v] = Ndot[s] * f;
            c->emitted[v] += Ndot[s] * f;
        }
    }
    CK(cudaStreamSynchronize(c->stream));
    cudaFree(c->d_src_g); cudaFree(c->d_src_S); c->d_src_g = nullptr; c->d_src_S = nullptr;
    cudaFree(c->d_blocked); c->d_blocked = nullptr; c->mask_level = -1;
    c->h_src_S = S;
    c->h_R.assign((size_t)nsrc, 0.0);
    c->h_nopen.assign((size_t)nsrc, -1.0);         // (-1: no mask, all root rays open)
    if (nsrc > 0) {
        CK(cudaMalloc(&c->d_src_g, g.size() * sizeof(double)));
        CK(cudaMalloc(&c->d_src_S, S.size() * sizeof(double)));
        CK(cudaMemcpy(c->d_src_g, g.data(), g.size() * sizeof(double), cudaMemcpyHostToDevice));
        CK(cudaMemcpy(c->d_src_S, S.data(), S.size() * sizeof(double), cudaMemcpyHostToDevice));
    }
    c->nsrc = nsrc;
    c->have_src = true;
    c->have_rates = false; c->have_accum = false; ++c->epoch;
    return ARC_OK;
}

int arc_get_thin_radii(arc_ctx *c, double *R_cells)
{
    if (!c) return ARC_EINVAL;
    if (!c->have_src) return fail(c, ARC_ESTATE, "arc_get_thin_radii: no sources set");
    if (!R_cells && c->nsrc > 0) return fail(c, ARC_EINVAL, "arc_get_thin_radii: NULL argument");
    for (int s = 0; s < c->nsrc; ++s) R_cells[s] = c->h_R[(size_t)s];
    return ARC_OK;
}

int arc_set_thin_radii(arc_ctx *c, const double *R_cells)
{
    if (!c) return ARC_EINVAL;
    if (!c->have_src) return fail(c, ARC_ESTATE, "arc_set_thin_radii: no sources set");
    if (!R_cells && c->nsrc > 0) return fail(c, ARC_EINVAL, "arc_set_thin_radii: NULL argument");
    for (int s = 0; s < c->nsrc; ++s)
        if (!(R_cells[s] >= 0.0) || !std::isfinite(R_cells[s])) return fail(c, ARC_EINVAL, "arc_set_thin_radii: radii must be finite and >= 0");
    for (int s = 0; s < c->nsrc; ++s) c->h_R[(size_t)s] = R_cells[s];
    c->have_rates = false; c->have_accum = false;
    return ARC_OK;
}

int arc_set_emission_mask(arc_ctx *c, const uint8_t *blocked, int level)
{
    if (!c) return ARC_EINVAL;
    if (!c->have_src) return fail(c, ARC_ESTATE, "arc_set_emission_mask: call arc_set_sources first");
    const int nb = c->spec.nb;
    CK(cudaStreamSynchronize(c->stream));
    cudaFree(c->d_blocked); c->d_blocked = nullptr; c->mask_level = -1;
    for (int v = 0; v < ARC_MAX_BINS; ++v) c->emitted[v] = 0.0;
    ++c->epoch;
    if (!blocked) {
        c->h_nopen.assign((size_t)c->nsrc, -1.0);
        for (int s = 0; s < c->nsrc; ++s) for (int v = 0; v < nb; ++v) c->emitted[v] += c->h_src_S[(size_t)s * nb + v];
        c->have_rates = false; c->have_accum = false;
        return ARC_OK;
    }
    if (level != c->p.l0) return fail(c, ARC_EINVAL, "arc_set_emission_mask: level must equal arc_params.l0");
    const size_t npix0 = (size_t)12 << (2 * level);
    for (int s = 0; s < c->nsrc; ++s) {
        size_t nopen = npix0;
        for (size_t p = 0; p < npix0; ++p) if (blocked[(size_t)s * npix0 + p]) --nopen;
        c->h_nopen[(size_t)s] = (double)nopen;
        for (int v = 0; v < nb; ++v) c->emitted[v] += c->h_src_S[(size_t)s * nb + v] / (double)npix0 * (double)nopen;
    }
    if (c->nsrc > 0) {
        CK(cudaMalloc(&c->d_blocked, (size_t)c->nsrc * npix0));
        CK(cudaMemcpy(c->d_blocked, blocked, (size_t)c->nsrc * npix0, cudaMemcpyHostToDevice));
    }
    c->mask_level = level;
    c->have_rates = false; c->have_accum = false;
    return ARC_OK;
}

}  // extern "C"
