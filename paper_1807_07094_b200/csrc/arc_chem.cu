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
#include <cmath>

namespace {

struct Coef {
    double aHII, aHeII, aHeIII;        // recombination [cm^3/s]
    double cHI, cHeI, cHeII;           // collisional ionisation [cm^3/s]
    double cool_rHII, cool_rHeII, cool_rHeIII;   // recombination cooling [erg cm^3/s]
    double cool_xHI, cool_xHeII;       // collisional excitation cooling
    double cool_ff;                    // bremsstrahlung
};

// The fits are products of powers of lambda_X = 2 T_X / T.  With L = ln T every such power is a constant times
// exp(-a L), and species that share an exponent share the exponential; (1 + u)^s = exp(s ln(1 + u)).  The constants
// (prefactor x (2 T_X)^a, (2 T_X / l0)^q) are evaluated once on the host (chem_consts) and passed by value: one
// sub-cycle costs 1 log + 1 reciprocal + 1 sqrt + 9 exp + 4 exp/log pairs (+ 8 exp and 3 pairs with collisional
// ionisation) instead of 16 exp, 4 pow and 4-8 log (25 exp, 7 pow, 4-11 log).  Same functions of T as DESIGN.md 2.1,
// to a few ulp.
struct ChemK {
    double p_rec, q_rec, s_rec, kH_rec, kB_rec, uH_rec, uB_rec;     // alpha_HII(lambda_H), alpha_HeIII = 2 alpha_HII(lambda_HeII)
    double p_cl, q_cl, s_cl, kH_cl, kB_cl, uH_cl, uB_cl;            // recombination cooling (x T), He III = 8 x at lambda_HeII
    double p_he, k_he;                                              // alpha_HeII radiative
    double kcHI, ucHI, kcHeI, ucHeI, kcHeII, ucHeII;                // collisional ionisation
    int coll, p_rec_is_15;
};

// e^x for the rate table, 3e-13 relative: x = k ln2 + r with |r| <= ln2 / 2 (two-part ln2), the Taylor polynomial of degree 10
// in Horner form, scaled by 2^k on the exponent field.  No special cases (the fits never pass it a NaN or more than +60;
// below e^-700 the result is 0: the fits multiply it by numbers of order 1e-10 .. 1e+2) - 19 instructions against the ~30 of
// the library's exp, which the table calls 18-26 times per sub-cycle.
__device__ __forceinline__ double exp_table(double x)
{
    const double MAGIC = 6755399441055744.0;                           // 1.5 * 2^52: round to nearest integer
    const double kt = fma(x, 1.4426950408889634074, MAGIC);
    const int k = __double2loint(kt);
    const double kd = kt - MAGIC;
    double r = fma(kd, -6.93147180369123816490e-01, x);
    r = fma(kd, -1.90821492927058770002e-10, r);
    double p = 1.0 / 3628800.0;
    p = fma(p, r, 1.0 / 362880.0);
    p = fma(p, r, 1.0 / 40320.0);
    p = fma(p, r, 1.0 / 5040.0);
    p = fma(p, r, 1.0 / 720.0);
    p = fma(p, r, 1.0 / 120.0);
    p = fma(p, r, 1.0 / 24.0);
    p = fma(p, r, 1.0 / 6.0);
    p = fma(p, r, 0.5);
    p = fma(p, r, 1.0);
    p = fma(p, r, 1.0);                                                // e^r in [0.707, 1.415]
    const double v = __hiloint2double(__double2hiint(p) + (k << 20), __double2loint(p));      // * 2^k
    return x < -700.0 ? 0.0 : v;
}

// ln x for the rate table (x = T >= 1 K or 1 + u >= 1: normal, positive), 1e-13 absolute: x = 2^e m with m in [0.707, 1.414],
// s = (m - 1)/(m + 1) from the hardware reciprocal seed and two Newton steps, ln m = 2 s (1 + s^2/3 + ... + s^14/15).
// 27 instructions against the ~40 of the library's log (denormals, NaN, infinities).
__device__ __forceinline__ double log_table(double x)
{
    int hi = __double2hiint(x);
    int e = (hi >> 20) - 1023;
    hi = (hi & 0x000fffff) | 0x3ff00000;
    const bool up = hi > 0x3ff6a09e;                                   // m > sqrt(2): use m / 2
    if (up) { hi -= 0x00100000; e += 1; }
    const double m = __hiloint2double(hi, __double2loint(x));
    const double f = m - 1.0, d = m + 1.0;
    double rc;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(rc) : "d"(d));             // ~20 bits; d in [1.7, 2.42]
    rc = fma(fma(-d, rc, 1.0), rc, rc);
    rc = fma(fma(-d, rc, 1.0), rc, rc);
    const double sq = f * rc, s2 = sq * sq;
    double p = 1.0 / 15.0;
    p = fma(p, s2, 1.0 / 13.0);
    p = fma(p, s2, 1.0 / 11.0);
    p = fma(p, s2, 1.0 / 9.0);
    p = fma(p, s2, 1.0 / 7.0);
    p = fma(p, s2, 1.0 / 5.0);
    p = fma(p, s2, 1.0 / 3.0);
    p = fma(p, s2, 1.0);
    return fma((double)e, 0.693147180559945309417, 2.0 * sq * p);
}

template <bool FAST> struct RtMath;
template <> struct RtMath<false> {
    static __device__ __forceinline__ double ex(double x) { return exp(x); }
    static __device__ __forceinline__ double lg(double x) { return log(x); }
};
template <> struct RtMath<true> {
    static __device__ __forceinline__ double ex(double x) { return exp_table(x); }
    static __device__ __forceinline__ double lg(double x) { return log_table(x); }
};

// FAST (the sub-cycled kernel, where the table is evaluated once per sub-cycle): the exponentials and logarithms of the fits
// from exp_table / log_table.  The once-per-cell users (isothermal kernel, time step) keep the library's functions.
template <bool FAST = false>
__device__ __forceinline__ void rate_table(double T, const ChemK &q, Coef &k)
{
    const double KB = 1.380649e-16;
    const double TR_H = 157807.0, TR_HE1 = 285335.0, TR_HE2 = 631515.0;   // ionisation thresholds in K
    auto exp = [](double x) { return RtMath<FAST>::ex(x); };             // (these shadow ::exp and ::log inside this function)
    auto log = [](double x) { return RtMath<FAST>::lg(x); };
    const double L = log(T), iT = 1.0 / T;
    // recombination and its cooling: A0 lambda^p / (1 + (lambda/l0)^q)^s
    const double ep = exp(-q.p_rec * L), eq = exp(-q.q_rec * L);
    k.aHII = q.kH_rec * ep * exp(-q.s_rec * log(1.0 + q.uH_rec * eq));
    k.aHeIII = q.kB_rec * ep * exp(-q.s_rec * log(1.0 + q.uB_rec * eq));
    const double Tm15 = q.p_rec_is_15 ? ep : exp(-1.5 * L);
    const double cp = T * exp(-q.p_cl * L), cq = exp(-q.q_cl * L);
    k.cool_rHII = q.kH_cl * cp * exp(-q.s_cl * log(1.0 + q.uH_cl * cq));
    k.cool_rHeIII = q.kB_cl * cp * exp(-q.s_cl * log(1.0 + q.uB_cl * cq));
    // dielectronic recombination of He II: e^{-470000/T} = (e^{-94000/T})^5
    const double w = exp(-94000.0 * iT), w2 = w * w;
    const double adi = 1.9e-3 * Tm15 * (w2 * w2 * w) * (1.0 + 0.3 * w);
    const double aHeII_rad = q.k_he * exp(-q.p_he * L);
    k.aHeII = aHeII_rad + adi;
    k.cool_rHeII = KB * T * aHeII_rad + 6.54e-11 * adi;
    k.cHI = k.cHeI = k.cHeII = 0.0;
    if (q.coll) {   // X T^-1.5 e^{-lambda/2} lambda^-a / (1 + (lambda/l0)^b)^c
        const double e1089 = exp(1.089 * L);
        k.cHI = q.kcHI * Tm15 * exp(-TR_H * iT) * e1089 * exp(-1.101 * log(1.0 + q.ucHI * exp(-0.874 * L)));
        k.cHeI = q.kcHeI * Tm15 * exp(-TR_HE1 * iT) * exp(1.146 * L) * exp(-1.056 * log(1.0 + q.ucHeI * exp(-0.987 * L)));
        k.cHeII = q.kcHeII * Tm15 * exp(-TR_HE2 * iT) * e1089 * exp(-1.275 * log(1.0 + q.ucHeII * exp(-0.735 * L)));
    }
    const double sqT = sqrt(T);
    const double damp = 1.0 / (1.0 + sqT * 3.1622776601683794e-3);        // 1 / (1 + sqrt(T / 1e5))
    k.cool_xHI = 7.5e-19 * exp(-118348.0 * iT) * damp;
    k.cool_xHeII = 5.54e-17 * exp(-0.397 * L - 473638.0 * iT) * damp;
    const double u = 5.5 - L * 0.43429448190325182765;       // 5.5 - log10 T
    k.cool_ff = 1.42e-27 * (1.1 + 0.34 * exp(-u * u / 3.0)) * sqT;
}

// host: the constants of the fits for the chosen recombination case
static ChemK chem_consts(bool caseB, bool coll)
{
    const double LH = 2.0 * 157807.0, LA = 2.0 * 285335.0, LB = 2.0 * 631515.0;
    ChemK q{};
    double A0, l0, C0, m0;
    if (caseB) { A0 = 2.753e-14; q.p_rec = 1.5; l0 = 2.74; q.q_rec = 0.407; q.s_rec = 2.242;
                 C0 = 3.435e-30; q.p_cl = 1.97; m0 = 2.25; q.q_cl = 0.376; q.s_cl = 3.72; q.k_he = 1.26e-14; q.p_he = 0.75; }
    else       { A0 = 1.269e-13; q.p_rec = 1.503; l0 = 0.522; q.q_rec = 0.47; q.s_rec = 1.923;
                 C0 = 1.778e-29; q.p_cl = 1.965; m0 = 0.541; q.q_cl = 0.502; q.s_cl = 2.697; q.k_he = 3.0e-14; q.p_he = 0.654; }
    q.kH_rec = A0 * std::pow(LH, q.p_rec); q.kB_rec = 2.0 * A0 * std::pow(LB, q.p_rec);
    q.uH_rec = std::pow(LH / l0, q.q_rec); q.uB_rec = std::pow(LB / l0, q.q_rec);
    q.kH_cl = C0 * std::pow(LH, q.p_cl); q.kB_cl = 8.0 * C0 * std::pow(LB, q.p_cl);
    q.uH_cl = std::pow(LH / m0, q.q_cl); q.uB_cl = std::pow(LB / m0, q.q_cl);
    q.k_he *= std::pow(LA, q.p_he);
    q.kcHI = 21.11 * std::pow(LH, -1.089); q.ucHI = std::pow(LH / 0.354, 0.874);
    q.kcHeI = 32.38 * std::pow(LA, -1.146); q.ucHeI = std::pow(LA / 0.416, 0.987);
    q.kcHeII = 19.95 * std::pow(LB, -1.089); q.ucHeII = std::pow(LB / 0.553, 0.735);
    q.coll = coll ? 1 : 0; q.p_rec_is_15 = q.p_rec == 1.5 ? 1 : 0;
    return q;
}

__device__ __forceinline__ double clamp01(double v, double lo) { return v < lo ? lo : (v > 1.0 ? 1.0 : v); }

// state of one cell during the sub-cycle loop
struct Cell {
    double nH, nHe, x0, x1, x2, T, G0, G1, G2, H0, H1, H2, t;
    int n;
};

// one sub-cycle of PAPER.md:136-154 (readings G12, G15-G17, G23, G24); k = rate table at c.T (ISO: evaluated by the caller)
template <bool ISO, bool FAST = false>
__device__ __forceinline__ void chem_subcycle(Cell &c, Coef &k, const ChemK &q, double dt, double eps, double x_floor, int max_sub)
{
    const double KB = 1.380649e-16;
    // collisional-ionisation cooling = threshold energy x rate (13.6, 24.6, 54.4 eV in erg)
    const double EI_H = 2.18e-11, EI_HE1 = 3.94e-11, EI_HE2 = 8.72e-11;
    const double nH = c.nH, nHe = c.nHe, x0 = c.x0, x1 = c.x1, x2 = c.x2;
    const double xHII = 1.0 - x0;
    double xHeIII = 1.0 - x1 - x2; if (xHeIII < 0.0) xHeIII = 0.0;
    const double ne = nH * xHII + nHe * (x2 + 2.0 * xHeIII);
    if (!ISO) rate_table<FAST>(c.T, q, k);
    // Eq. 4 written as Eq. 5 (dn/dt = D - C n), in fractions
    const double C0 = c.G0 + k.cHI * ne,              D0 = k.aHII * ne * xHII;
    const double C1 = c.G1 + k.cHeI * ne,             D1 = k.aHeII * ne * x2;
    const double C2 = (c.G2 + k.cHeII * ne) + k.aHeII * ne;
    const double D2 = (c.G1 + k.cHeI * ne) * x1 + k.aHeIII * ne * xHeIII;
    double left = dt - c.t, dts = left;
    double heat = 0.0, cool = 0.0, E = 0.0;
    if (!ISO) {
        const double nHI = nH * x0, nHeI = nHe * x1, nHeII = nHe * x2, nHII = nH * xHII, nHeIII = nHe * xHeIII;
        heat = (c.H0 * nHI + c.H1 * nHeI) + c.H2 * nHeII;
        cool = ne * (k.cool_rHII * nHII + k.cool_rHeII * nHeII + k.cool_rHeIII * nHeIII
                     + EI_H * k.cHI * nHI + EI_HE1 * k.cHeI * nHeI + EI_HE2 * k.cHeII * nHeII
                     + k.cool_xHI * nHI + k.cool_xHeII * nHeII
                     + k.cool_ff * (nHII + nHeII + 4.0 * nHeIII));
        E = 1.5 * KB * c.T * (nH + nHe + ne);
    }
    if (c.n != max_sub - 1) {
        const double xdot = D0 - C0 * x0;
        if (xdot != 0.0) dts = fmin(dts, eps * x0 / fabs(xdot));
        if (!ISO && heat - cool != 0.0) dts = fmin(dts, eps * E / fabs(heat - cool));
    }
    const double y0 = (x0 + D0 * dts) / (1.0 + C0 * dts);                     // Eq. 5 backward difference
    const double y1 = (x1 + D1 * dts) / (1.0 + C1 * dts);
    const double y2 = (x2 + D2 * dts) / (1.0 + C2 * dts);
    c.x0 = clamp01(y0, x_floor); c.x1 = clamp01(y1, x_floor); c.x2 = clamp01(y2, 0.0);
    if (c.x1 + c.x2 > 1.0) { const double s = c.x1 + c.x2; c.x1 = c.x1 / s; c.x2 = c.x2 / s; }
    if (!ISO) {
        const double En = (E + heat * dts) / (1.0 + (cool / E) * dts);
        double xHeIII_n = 1.0 - c.x1 - c.x2; if (xHeIII_n < 0.0) xHeIII_n = 0.0;
        const double ne_n = nH * (1.0 - c.x0) + nHe * (c.x2 + 2.0 * xHeIII_n);
        c.T = fmax(En / (1.5 * KB * (nH + nHe + ne_n)), 1.0);
    }
    c.t = (dts >= left) ? dt : c.t + dts;
    ++c.n;
}

template <typename FT, bool ISO>
__device__ __forceinline__ void chem_load(Cell &c, long long i, long long ncell, double Yp, const FT *__restrict__ nHf,
                                          const FT *__restrict__ xHIf, const FT *__restrict__ xHeIf, const FT *__restrict__ xHeIIf,
                                          const FT *__restrict__ Tf, const double *__restrict__ rates)
{
    c.nH = (double)nHf[i];
    c.nHe = c.nH * Yp / (4.0 * (1.0 - Yp));
    c.x0 = (double)xHIf[i]; c.x1 = (double)xHeIf[i]; c.x2 = (double)xHeIIf[i]; c.T = (double)Tf[i];
    c.G0 = rates[i]; c.G1 = rates[ncell + i]; c.G2 = rates[2 * ncell + i];
    c.H0 = c.H1 = c.H2 = 0.0;
    if (!ISO) { c.H0 = rates[3 * ncell + i]; c.H1 = rates[4 * ncell + i]; c.H2 = rates[5 * ncell + i]; }
    c.t = 0.0; c.n = 0;
}

// Isothermal runs (configs 1-2): the rate table does not change during the call and a sub-cycle is a few dozen flops,
// so one thread keeps one cell; fully coalesced grid-stride pass.
template <typename FT>
__global__ void __launch_bounds__(128) arc_chem_iso_kernel(long long ncell, double dt, double Yp, double eps, double x_floor,
                                                          int max_sub, ChemK q,
                                                          const FT *__restrict__ nHf, FT *__restrict__ xHIf, FT *__restrict__ xHeIf,
                                                          FT *__restrict__ xHeIIf, FT *__restrict__ Tf,
                                                          const double *__restrict__ rates, DevStats *stats, const SchedState *__restrict__ sc)
{
    if (sc->error != ARC_DEV_OK || sc->in_flight != 0) return;      // the last trace aborted (async mode): fields stay as they are
    unsigned long long my_sub = 0; unsigned int my_max = 0;
    // an isothermal box usually has ONE temperature: the table at the block's first cell is evaluated once (first warp)
    // and shared; a cell at another temperature evaluates its own (same function, same argument: same bits)
    __shared__ Coef s_k;
    __shared__ double s_T;
    {
        const long long first = blockIdx.x * (long long)blockDim.x;
        if (threadIdx.x < 32) {
            Coef k0;
            const double T0 = (double)Tf[first < ncell ? first : 0];
            rate_table(T0, q, k0);
            if (threadIdx.x == 0) { s_k = k0; s_T = T0; }
        }
        __syncthreads();
    }
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < ncell; i += (long long)gridDim.x * blockDim.x) {
        Cell c; Coef k;
        chem_load<FT, true>(c, i, ncell, Yp, nHf, xHIf, xHeIf, xHeIIf, Tf, rates);
        if (c.T == s_T) k = s_k; else rate_table(c.T, q, k);
        while (c.t < dt && c.n < max_sub) chem_subcycle<true>(c, k, q, dt, eps, x_floor, max_sub);
        xHIf[i] = (FT)c.x0; xHeIf[i] = (FT)c.x1; xHeIIf[i] = (FT)c.x2;
        my_sub += (unsigned long long)c.n;
        my_max = max(my_max, (unsigned int)c.n);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        my_sub += __shfl_xor_sync(0xffffffffu, my_sub, o);
        my_max = max(my_max, __shfl_xor_sync(0xffffffffu, my_max, o));
    }
    if ((threadIdx.x & 31) == 0) { atomicAdd(&stats->subcycles, my_sub); atomicAdd(&stats->subcycles_total, my_sub); atomicMax(&stats->max_sub, my_max); }
}

// Evolving temperature: every sub-cycle re-evaluates the rate table (a few thousand fp64 instructions) and the number of
// sub-cycles per cell runs from 1 (most of the box) to max_sub (ionisation fronts), so a lane that kept its cell until
// the slowest cell of the warp finished would idle most of the time.  Persistent warps instead: every lane owns one
// cell; each warp iteration runs ONE sub-cycle on every lane, and lanes whose cell is finished write it back and take
// the next cells from a global counter (one atomicAdd per warp and refill) - all 32 lanes stay busy until the grid is
// used up.  The arithmetic per cell is exactly that of the one-thread-per-cell loop.
// 5 blocks per SM (96 registers, no spills): measured best of 4 / 5 / 6 / 8 (128 / 96 / 80 / 64 registers) on configs 3, 4.
template <typename FT>
__global__ void __launch_bounds__(128, 5) arc_chem_kernel(long long ncell, double dt, double Yp, double eps, double x_floor,
                                                      int max_sub, ChemK q,
                                                      const FT *__restrict__ nHf, FT *__restrict__ xHIf, FT *__restrict__ xHeIf,
                                                      FT *__restrict__ xHeIIf, FT *__restrict__ Tf,
                                                      const double *__restrict__ rates, DevStats *stats, const SchedState *__restrict__ sc)
{
    if (sc->error != ARC_DEV_OK || sc->in_flight != 0) return;      // the last trace aborted (async mode): fields stay as they are
    const unsigned lane = threadIdx.x & 31u;
    unsigned long long my_sub = 0; unsigned int my_max = 0;
    long long mine = -1;                          // this lane's cell, -1 = none
    bool drained = false;                         // warp-uniform: the counter has passed ncell
    Cell c; Coef k;
    c.n = 0; c.t = 0.0;
    for (;;) {
        const unsigned idle = __ballot_sync(0xffffffffu, mine < 0);
        if (idle != 0u && !drained) {
            const int want = __popc(idle);
            long long base = 0;
            if (lane == 0) base = (long long)atomicAdd(&stats->chem_next, (unsigned long long)want);
            base = __shfl_sync(0xffffffffu, base, 0);
            drained = base + want >= ncell;
            if (mine < 0) {
                const long long i = base + __popc(idle & ((1u << lane) - 1u));
                if (i < ncell) { mine = i; chem_load<FT, false>(c, i, ncell, Yp, nHf, xHIf, xHeIf, xHeIIf, Tf, rates); }
            }
        }
        if (__all_sync(0xffffffffu, mine < 0)) break;
        if (mine >= 0) {
            if (c.t < dt && c.n < max_sub) chem_subcycle<false, true>(c, k, q, dt, eps, x_floor, max_sub);
            if (!(c.t < dt && c.n < max_sub)) {
                xHIf[mine] = (FT)c.x0; xHeIf[mine] = (FT)c.x1; xHeIIf[mine] = (FT)c.x2; Tf[mine] = (FT)c.T;
                my_sub += (unsigned long long)c.n;
                my_max = max(my_max, (unsigned int)c.n);
                mine = -1;
            }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        my_sub += __shfl_xor_sync(0xffffffffu, my_sub, o);
        my_max = max(my_max, __shfl_xor_sync(0xffffffffu, my_max, o));
    }
    if (lane == 0) { atomicAdd(&stats->subcycles, my_sub); atomicAdd(&stats->subcycles_total, my_sub); atomicMax(&stats->max_sub, my_max); }
}

// Radiative-transfer time step (include/arc.h arc_suggest_dt): one streaming pass, 28 B per cell
// (five fields at the field dtype + Gamma_HI), minimum by warp shuffles and one 64-bit atomicMin per warp on the bits of
// the (positive) double.  The tau > 0.5 test is products only, in the oracle's order: the same cells qualify.
template <typename FT>
__global__ void __launch_bounds__(256) arc_dt_kernel(long long ncell, int scheme, double eps, double sigma1, double d, double Yp,
                                                    ChemK q, const FT *__restrict__ nHf, const FT *__restrict__ xHIf,
                                                    const FT *__restrict__ xHeIf, const FT *__restrict__ xHeIIf, const FT *__restrict__ Tf,
                                                    const double *__restrict__ GammaHI, unsigned long long *out, const SchedState *__restrict__ sc)
{
    if (sc->error != ARC_DEV_OK || sc->in_flight != 0) return;
    double best = __longlong_as_double(0x7ff0000000000000ll);
    unsigned long long used = 0;
    for (long long c = blockIdx.x * (long long)blockDim.x + threadIdx.x; c < ncell; c += (long long)gridDim.x * blockDim.x) {
        const double nH = (double)nHf[c], x0 = (double)xHIf[c], x1 = (double)xHeIf[c], x2 = (double)xHeIIf[c];
        const double nHe = nH * Yp / (4.0 * (1.0 - Yp));
        const double xHII = 1.0 - x0;
        double xHeIII = 1.0 - x1 - x2; if (xHeIII < 0.0) xHeIII = 0.0;
        const double ne = nH * xHII + nHe * (x2 + 2.0 * xHeIII);
        Coef k;
        rate_table((double)Tf[c], q, k);
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
    arc_dt_kernel<FT><<<(int)(nb < cap ? nb : cap), 256, 0, c->stream>>>(c->ncell, scheme, eps, c->spec.sig[0][0], c->dx, c->p.Yp,
                                                                        chem_consts(c->p.caseB != 0, c->p.coll_ion != 0), f[0], f[1], f[2], f[3], f[4], c->d_rates, c->d_dt, c->d_sched);
    ++c->launches;
    return cudaGetLastError();
}

template <typename FT>
cudaError_t launch_chem(arc_ctx *c, double dt)
{
    FT **f = reinterpret_cast<FT **>(c->f);
    const ChemK q = chem_consts(c->p.caseB != 0, c->p.coll_ion != 0);
    const long long nb = (c->ncell + 127) / 128;
    if (c->p.isothermal) {
        // exactly the co-resident blocks, grid-stride: every block evaluates the rate table once (a chain of a thousand
        // dependent fp64 instructions), so blocks beyond one wave would only repeat that latency
        int per_sm = 0;
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, arc_chem_iso_kernel<FT>, 128, 0);
        if (e != cudaSuccess) return e;
        const long long cap = (long long)c->n_sm * (per_sm > 0 ? per_sm : 1);
        arc_chem_iso_kernel<FT><<<(int)(nb < cap ? nb : cap), 128, 0, c->stream>>>(c->ncell, dt, c->p.Yp, c->p.eps_sub, c->p.x_floor, c->p.max_subcycles,
                                                                                 q, f[0], f[1], f[2], f[3], f[4], c->d_rates, c->d_stats, c->d_sched);
    } else {
        // persistent: exactly the co-resident blocks (stats->chem_next is zeroed by arc_update_chemistry)
        int per_sm = 0;
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, arc_chem_kernel<FT>, 128, 0);
        if (e != cudaSuccess) return e;
        const long long cap = (long long)c->n_sm * (per_sm > 0 ? per_sm : 1);
        arc_chem_kernel<FT><<<(int)(nb < cap ? nb : cap), 128, 0, c->stream>>>(c->ncell, dt, c->p.Yp, c->p.eps_sub, c->p.x_floor, c->p.max_subcycles,
                                                                             q, f[0], f[1], f[2], f[3], f[4], c->d_rates, c->d_stats, c->d_sched);
    }
    ++c->launches;
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
