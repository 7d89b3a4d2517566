// arc_chem.cu -- per-cell ionisation / heating update (Eq. 4-5, 166-172).
//
// One thread per cell; the five SoA fields and the six per-absorber rates are read fully coalesced, the
// sub-cycle loop runs in registers in fp64, the four evolving fields are written back at the field dtype.
// Every species obeys  dn/dt = D - C n  (Eq. 5) and is advanced by the backward difference
//      n <- (n + D dts) / (1 + C dts),
// with the sub-step dts = min(eps E/|dE/dt|, eps n_HI/|dn_HI/dt|, time left), eps = 0.1.
// Photo-rates per absorber are held fixed during the call.  Readings G12, G15-G17 of
// three absorbers with x_HeIII by closure, Jacobi order, E = 3/2 k T (n_H + n_He + n_e).
//
// Rate coefficients (reading G11): the paper takes them from Hui & Gnedin (1997) and
// prints only what fixes alpha_B(1e4 K) = 2.59e-13.  The fits below are the published
// Hui & Gnedin (1997) / Cen (1992) forms, typed here from DESIGN.md "Rate table", in lambda = 2 T_TR / T.
#include "arc_internal.cuh"

namespace {

struct Coef {
    double aHII, aHeII, aHeIII;        // recombination [cm^3/s]
    double cHI, cHeI, cHeII;           // collisional ionisation [cm^3/s]
    double cool_rHII, cool_rHeII, cool_rHeIII;   // recombination cooling [erg cm^3/s]
    double cool_xHI, cool_xHeII;       // collisional excitation cooling
    double cool_ff;                    // bremsstrahlung
};

// x^a for x > 0 through one log and one exp
__device__ __forceinline__ double powl_(double lnx, double a) { return exp(a * lnx); }

__device__ void rate_table(double T, bool caseB, bool coll, Coef &k)
{
    const double KB = 1.380649e-16;
    const double TR_H = 157807.0, TR_HE1 = 285335.0, TR_HE2 = 631515.0;   // ionisation thresholds in K
    const double lamH = 2.0 * TR_H / T, lamA = 2.0 * TR_HE1 / T, lamB = 2.0 * TR_HE2 / T;
    const double lnH = log(lamH), lnA = log(lamA), lnB = log(lamB), lnT = log(T);
    if (caseB) {
        k.aHII = 2.753e-14 * powl_(lnH, 1.5) / pow(1.0 + powl_(lnH - log(2.74), 0.407), 2.242);
        k.aHeII = 1.26e-14 * powl_(lnA, 0.75);
        k.aHeIII = 2.0 * 2.753e-14 * powl_(lnB, 1.5) / pow(1.0 + powl_(lnB - log(2.74), 0.407), 2.242);
        k.cool_rHII = 3.435e-30 * T * powl_(lnH, 1.97) / pow(1.0 + powl_(lnH - log(2.25), 0.376), 3.72);
        k.cool_rHeIII = 8.0 * 3.435e-30 * T * powl_(lnB, 1.97) / pow(1.0 + powl_(lnB - log(2.25), 0.376), 3.72);
    } else {
        k.aHII = 1.269e-13 * powl_(lnH, 1.503) / pow(1.0 + powl_(lnH - log(0.522), 0.47), 1.923);
        k.aHeII = 3.0e-14 * powl_(lnA, 0.654);
        k.aHeIII = 2.0 * 1.269e-13 * powl_(lnB, 1.503) / pow(1.0 + powl_(lnB - log(0.522), 0.47), 1.923);
        k.cool_rHII = 1.778e-29 * T * powl_(lnH, 1.965) / pow(1.0 + powl_(lnH - log(0.541), 0.502), 2.697);
        k.cool_rHeIII = 8.0 * 1.778e-29 * T * powl_(lnB, 1.965) / pow(1.0 + powl_(lnB - log(0.541), 0.502), 2.697);
    }
    // dielectronic recombination of He II
    const double Tm15 = exp(-1.5 * lnT);
    const double adi = 1.9e-3 * Tm15 * exp(-470000.0 / T) * (1.0 + 0.3 * exp(-94000.0 / T));
    const double aHeII_rad = k.aHeII;
    k.aHeII = aHeII_rad + adi;
    k.cool_rHeII = KB * T * aHeII_rad + 6.54e-11 * adi;
    k.cHI = k.cHeI = k.cHeII = 0.0;
    if (coll) {
        k.cHI = 21.11 * Tm15 * exp(-0.5 * lamH) * powl_(lnH, -1.089) / pow(1.0 + powl_(lnH - log(0.354), 0.874), 1.101);
        k.cHeI = 32.38 * Tm15 * exp(-0.5 * lamA) * powl_(lnA, -1.146) / pow(1.0 + powl_(lnA - log(0.416), 0.987), 1.056);
        k.cHeII = 19.95 * Tm15 * exp(-0.5 * lamB) * powl_(lnB, -1.089) / pow(1.0 + powl_(lnB - log(0.553), 0.735), 1.275);
    }
    const double damp = 1.0 / (1.0 + sqrt(T / 1.0e5));
    k.cool_xHI = 7.5e-19 * exp(-118348.0 / T) * damp;
    k.cool_xHeII = 5.54e-17 * exp(-0.397 * lnT) * exp(-473638.0 / T) * damp;
    const double u = 5.5 - lnT * 0.43429448190325182765;     // 5.5 - log10 T
    k.cool_ff = 1.42e-27 * (1.1 + 0.34 * exp(-u * u / 3.0)) * sqrt(T);
}

__device__ __forceinline__ double clamp01(double v, double lo) { return v < lo ? lo : (v > 1.0 ? 1.0 : v); }

template <typename FT, bool ISO>
__global__ void __launch_bounds__(128) arc_chem_kernel(long long ncell, double dt, double Yp, double eps, double x_floor,
                                                      int max_sub, int caseB, int coll,
                                                      const FT *__restrict__ nHf, FT *__restrict__ xHIf, FT *__restrict__ xHeIf,
                                                      FT *__restrict__ xHeIIf, FT *__restrict__ Tf,
                                                      const double *__restrict__ rates, DevStats *stats)
{
    const double KB = 1.380649e-16;
    // collisional-ionisation cooling = threshold energy x rate (13.6, 24.6, 54.4 eV in erg)
    const double EI_H = 2.18e-11, EI_HE1 = 3.94e-11, EI_HE2 = 8.72e-11;
    unsigned long long my_sub = 0; unsigned int my_max = 0;
    for (long long c = blockIdx.x * (long long)blockDim.x + threadIdx.x; c < ncell; c += (long long)gridDim.x * blockDim.x) {
        const double nH = (double)nHf[c];
        const double nHe = nH * Yp / (4.0 * (1.0 - Yp));
        double x0 = (double)xHIf[c], x1 = (double)xHeIf[c], x2 = (double)xHeIIf[c], T = (double)Tf[c];
        const double G0 = rates[c], G1 = rates[ncell + c], G2 = rates[2 * ncell + c];
        double H0 = 0.0, H1 = 0.0, H2 = 0.0;
        if (!ISO) { H0 = rates[3 * ncell + c]; H1 = rates[4 * ncell + c]; H2 = rates[5 * ncell + c]; }
        Coef k;
        if (ISO) rate_table(T, caseB != 0, coll != 0, k);
        double t = 0.0;
        int n = 0;
        while (t < dt && n < max_sub) {
            const double xHII = 1.0 - x0;
            double xHeIII = 1.0 - x1 - x2; if (xHeIII < 0.0) xHeIII = 0.0;
            const double ne = nH * xHII + nHe * (x2 + 2.0 * xHeIII);
            if (!ISO) rate_table(T, caseB != 0, coll != 0, k);
            // Eq. 4 written as Eq. 5 (dn/dt = D - C n), in fractions
            const double C0 = G0 + k.cHI * ne,              D0 = k.aHII * ne * xHII;
            const double C1 = G1 + k.cHeI * ne,             D1 = k.aHeII * ne * x2;
            const double C2 = (G2 + k.cHeII * ne) + k.aHeII * ne;
            const double D2 = (G1 + k.cHeI * ne) * x1 + k.aHeIII * ne * xHeIII;
            double left = dt - t, dts = left;
            double heat = 0.0, cool = 0.0, E = 0.0;
            if (!ISO) {
                const double nHI = nH * x0, nHeI = nHe * x1, nHeII = nHe * x2, nHII = nH * xHII, nHeIII = nHe * xHeIII;
                heat = (H0 * nHI + H1 * nHeI) + H2 * nHeII;
                cool = ne * (k.cool_rHII * nHII + k.cool_rHeII * nHeII + k.cool_rHeIII * nHeIII
                             + EI_H * k.cHI * nHI + EI_HE1 * k.cHeI * nHeI + EI_HE2 * k.cHeII * nHeII
                             + k.cool_xHI * nHI + k.cool_xHeII * nHeII
                             + k.cool_ff * (nHII + nHeII + 4.0 * nHeIII));
                E = 1.5 * KB * T * (nH + nHe + ne);
            }
            if (n != max_sub - 1) {
                const double xdot = D0 - C0 * x0;
                if (xdot != 0.0) dts = fmin(dts, eps * x0 / fabs(xdot));
                if (!ISO && heat - cool != 0.0) dts = fmin(dts, eps * E / fabs(heat - cool));
            }
            const double y0 = (x0 + D0 * dts) / (1.0 + C0 * dts);                     // Eq. 5 backward difference
            const double y1 = (x1 + D1 * dts) / (1.0 + C1 * dts);
            const double y2 = (x2 + D2 * dts) / (1.0 + C2 * dts);
            x0 = clamp01(y0, x_floor); x1 = clamp01(y1, x_floor); x2 = clamp01(y2, 0.0);
            if (x1 + x2 > 1.0) { const double s = x1 + x2; x1 = x1 / s; x2 = x2 / s; }
            if (!ISO) {
                const double En = (E + heat * dts) / (1.0 + (cool / E) * dts);
                double xHeIII_n = 1.0 - x1 - x2; if (xHeIII_n < 0.0) xHeIII_n = 0.0;
                const double ne_n = nH * (1.0 - x0) + nHe * (x2 + 2.0 * xHeIII_n);
                T = fmax(En / (1.5 * KB * (nH + nHe + ne_n)), 1.0);
            }
            t = (dts >= left) ? dt : t + dts;
            ++n;
        }
        xHIf[c] = (FT)x0; xHeIf[c] = (FT)x1; xHeIIf[c] = (FT)x2;
        if (!ISO) Tf[c] = (FT)T;
        my_sub += (unsigned long long)n;
        my_max = max(my_max, (unsigned int)n);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        my_sub += __shfl_xor_sync(0xffffffffu, my_sub, o);
        my_max = max(my_max, __shfl_xor_sync(0xffffffffu, my_max, o));
    }
    if ((threadIdx.x & 31) == 0) { atomicAdd(&stats->subcycles, my_sub); atomicMax(&stats->max_sub, my_max); }
}

// Radiative-transfer time step (include/arc.h arc_suggest_dt): one streaming pass, 28 B per cell
// (five fields at the field dtype + Gamma_HI), minimum by warp shuffles and one 64-bit atomicMin per warp on the bits of
// the (positive) double.  The tau > 0.5 test is products only, in the oracle's order: the same cells qualify.
template <typename FT>
__global__ void __launch_bounds__(256) arc_dt_kernel(long long ncell, int scheme, double eps, double sigma1, double d, double Yp,
                                                    int caseB, int coll, const FT *__restrict__ nHf, const FT *__restrict__ xHIf,
                                                    const FT *__restrict__ xHeIf, const FT *__restrict__ xHeIIf, const FT *__restrict__ Tf,
                                                    const double *__restrict__ GammaHI, unsigned long long *out)
{
    double best = __longlong_as_double(0x7ff0000000000000ll);
    unsigned long long used = 0;
    for (long long c = blockIdx.x * (long long)blockDim.x + threadIdx.x; c < ncell; c += (long long)gridDim.x * blockDim.x) {
        const double nH = (double)nHf[c], x0 = (double)xHIf[c], x1 = (double)xHeIf[c], x2 = (double)xHeIIf[c];
        const double nHe = nH * Yp / (4.0 * (1.0 - Yp));
        const double xHII = 1.0 - x0;
        double xHeIII = 1.0 - x1 - x2; if (xHeIII < 0.0) xHeIII = 0.0;
        const double ne = nH * xHII + nHe * (x2 + 2.0 * xHeIII);
        Coef k;
        rate_table((double)Tf[c], caseB != 0, coll != 0, k);
        const double C0 = GammaHI[c] + k.cHI * ne, D0 = k.aHII * ne * xHII;
        const double nHI = __dmul_rn(nH, x0);
        const double ndot = fabs(nH * (D0 - C0 * x0));
        if (ndot == 0.0) continue;
        double dt;
        if (scheme == ARC_DT_NEUTRAL) {
            const double tau = __dmul_rn(__dmul_rn(nHI, sigma1), d);
            if (!(tau > 0.5)) continue;
            dt = eps * nHI / ndot;
        } else dt = eps / ((sigma1 * d) * ndot);
        ++used;
        best = fmin(best, dt);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        best = fmin(best, __shfl_xor_sync(0xffffffffu, best, o));
        used += __shfl_xor_sync(0xffffffffu, used, o);
    }
    if ((threadIdx.x & 31) == 0 && used) {
        atomicMin(out, (unsigned long long)__double_as_longlong(best));
        atomicAdd(out + 1, used);
    }
}

template <typename FT>
cudaError_t launch_dt(arc_ctx *c, int scheme, double eps)
{
    const long long nb = (c->ncell + 255) / 256;
    const long long cap = (long long)c->n_sm * 8;
    FT **f = reinterpret_cast<FT **>(c->f);
    arc_dt_kernel<FT><<<(int)(nb < cap ? nb : cap), 256, 0, c->stream>>>(c->ncell, scheme, eps, c->spec.sig[0][0], c->dx, c->p.Yp, c->p.caseB,
                                                                        c->p.coll_ion, f[0], f[1], f[2], f[3], f[4], c->d_rates, c->d_dt);
    return cudaGetLastError();
}

template <typename FT>
cudaError_t launch_chem(arc_ctx *c, double dt)
{
    const long long nb = (c->ncell + 127) / 128;
    const long long cap = (long long)c->n_sm * 32;
    const int grid = (int)(nb < cap ? nb : cap);
    FT **f = reinterpret_cast<FT **>(c->f);
    if (c->p.isothermal)
        arc_chem_kernel<FT, true><<<grid, 128, 0, c->stream>>>(c->ncell, dt, c->p.Yp, c->p.eps_sub, c->p.x_floor, c->p.max_subcycles,
                                                              c->p.caseB, c->p.coll_ion, f[0], f[1], f[2], f[3], f[4], c->d_rates, c->d_stats);
    else
        arc_chem_kernel<FT, false><<<grid, 128, 0, c->stream>>>(c->ncell, dt, c->p.Yp, c->p.eps_sub, c->p.x_floor, c->p.max_subcycles,
                                                               c->p.caseB, c->p.coll_ion, f[0], f[1], f[2], f[3], f[4], c->d_rates, c->d_stats);
    return cudaGetLastError();
}

}  // namespace

cudaError_t arc_launch_suggest_dt(arc_ctx *c, int scheme, double eps)
{
    return c->dtype == ARC_F32 ? launch_dt<float>(c, scheme, eps) : launch_dt<double>(c, scheme, eps);
}

cudaError_t arc_launch_chemistry(arc_ctx *c, double dt)
{
    return c->dtype == ARC_F32 ? launch_chem<float>(c, dt) : launch_chem<double>(c, dt);
}
