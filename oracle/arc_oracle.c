/* oracle/arc_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, single-threaded, fp64 implementation of the hot path of ARC
 * (Hartley & Ricotti 2018, arXiv:1807.07094): photon-conserving, spatially adaptive HEALPix
 * ray tracing from point sources through a uniform N^3 grid (Eq. 1),
 * the per-cell rate finalisation (Eq. 1) and the sub-cycled backward-
 * difference chemistry/thermal update (Eq. 4-5, 166-172).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
 * use it.  It shares no code with the CUDA path (paper_1807_07094_b200/csrc): both are typed
 * independently from DESIGN.md's arithmetic contract (sections "Readings" and "Contract").
 *
 * The method's result is DEFINED by the algorithm (which cells each ray visits, where it
 * splits), so the oracle is the algorithm, step by step, in the paper's order.  No blocking,
 * fusion or reordering: one explicit stack of ray records, depth first, one source at a time.
 *
 * Pins (tests/test_oracle_*.py): HEALPix ring-scheme closed form, own sincos vs libm,
 * brute-force line sampling of cell sequences, exact attenuation on axis-aligned rays, photon
 * conservation to 1e-10, partition of unity of the species weights, BDF closed forms, the
 * analytic Stromgren radius/growth.
 * Rate table (PAPER.md:162,172 cite Hui & Gnedin 1997; Fig. 2 is an image only): alpha_B(1e4 K) = 2.59e-13 is
 * the paper's; the recombination coefficients and the recombination cooling are pinned against the
 * standard tabulated values (tests/golden/textbook_rates.txt), He III by the hydrogenic scaling, collisional
 * ionisation against Voronov's (1997) independent fit (within 25 %), collisional-excitation cooling by its Lyman-alpha
 * thresholds (3/4 of the ionisation energies) and against the textbook collision strengths (25 % for H I, a factor two
 * for He II - the classic fit is no better than that), free-free against the textbook emissivity and Gaunt-factor
 * range, dielectronic recombination against the published fit parameters and the 40.8 eV core excitation.
 * Chemistry (tests/test_oracle_chem_pins.py): n_e against PAPER.md:73 in n_b, A_H, A_He; every term of the H I / He I /
 * He II backward differences (one-step identity + conservation of helium nuclei + closed-form equilibrium and cascade);
 * the energy update, T(E) and the sub-cycle limiter (one-step identities in states that isolate each cooling process,
 * mu by hand, convergence to scipy's integration of Eq. 4 + the energy equation, thermal-equilibrium root).
 * PARITY UNPINNED: nothing by structure; by VALUE the textbook numbers in tests/golden/textbook_rates.txt were typed
 * from outside this container (labelled there), and the He II excitation magnitude is only pinned to a factor two.
 *
 * Build: gcc -O2 -ffp-contract=off -fno-fast-math -shared -fPIC arc_oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_MAXNB 8
#define ORC_MAXLEVEL 16

/* pi rounded to double = 0x400921FB54442D18 (contract C1) */
static const double ORC_PI = 3.14159265358979323846;

enum { ORC_END_SPLIT = 0, ORC_END_DEPLETED = 1, ORC_END_ESCAPED = 2 };

typedef struct {
    int32_t N;
    int32_t field_dtype;      /* 0 = f32 fields (opacity rounded to f32), 1 = f64 */
    double box_cm;
    int32_t l0;               /* initial HEALPix level */
    int32_t Lmax;             /* rays at Lmax never split */
    double Phi;               /* rays per cell */
    double tau_term;          /* reading G7 */
    double Yp;                /* helium mass fraction */
    int32_t isothermal;
    int32_t caseB;
    int32_t coll_ion;
    int32_t max_subcycles;
    double eps_sub;
    double x_floor;
    int32_t geom_corr;        /* 0 none, 1 f_c (Eq. 2), 2 f_c + secondary f'_c (Eq. 3), 3 f_c squared */
    int32_t pad_;
    double thin_tau;          /* optical depth (softest bin) below which a source's surroundings count as
                                 optically thin, 0.1 in the paper; 0 = the approximation is off */
} orc_params;

typedef struct {
    uint64_t segments;
    uint64_t rays;
    uint64_t digest;
    uint64_t max_stack;
    uint64_t splits[ORC_MAXLEVEL];
    uint64_t rays_level[ORC_MAXLEVEL];
    uint64_t ends[3];
    double emitted[ORC_MAXNB];
    double absorbed[ORC_MAXNB];
    double escaped[ORC_MAXNB];
} orc_stats;

/* optional per-ray log (small configs only) */
typedef struct {
    int64_t cap_rays, cap_cells;
    int64_t n_rays, n_cells;
    int32_t *src; int32_t *level; int64_t *pix; int32_t *end; int64_t *first; int32_t *count;
    double *r_end;      /* radius at which the ray ended (grid units) */
    int32_t *cells;     /* linear cell index per segment */
    double *ds;         /* segment length per segment (grid units) */
} orc_raylog;

/* ------------------------------------------------------------------------------------------
 * O1. HEALPix nested pixel -> ring coordinates (Gorski et al. 2005, cited PAPER.md:45, 88).
 * z = zn/zd (exact integers), phi = m*pi/(4*nr) with integer m in [0, 8nr).
 * ------------------------------------------------------------------------------------------ */
static uint64_t take_bits(uint64_t v, int start)   /* bits start, start+2, start+4, ... packed */
{
    uint64_t r = 0;
    for (int b = 0; b < 32; ++b) r |= ((v >> (2 * b + start)) & 1ull) << b;
    return r;
}

void orc_pix2ring(int level, uint64_t pix, int64_t *zn, int64_t *zd, int64_t *m, int64_t *nr_out)
{
    static const int64_t R[12] = {2, 2, 2, 2, 3, 3, 3, 3, 4, 4, 4, 4};
    static const int64_t P[12] = {1, 3, 5, 7, 0, 2, 4, 6, 1, 3, 5, 7};
    const int64_t ns = (int64_t)1 << level;
    const uint64_t npface = (uint64_t)ns * (uint64_t)ns;
    const int f = (int)(pix >> (2 * level));
    const uint64_t q = pix & (npface - 1);
    const int64_t ix = (int64_t)take_bits(q, 0);
    const int64_t iy = (int64_t)take_bits(q, 1);
    const int64_t jr = R[f] * ns - ix - iy - 1;
    int64_t nr, k;
    if (jr < ns) {                 /* north polar cap */
        nr = jr; k = 0;
        *zn = 3 * ns * ns - nr * nr; *zd = 3 * ns * ns;
    } else if (jr > 3 * ns) {      /* south polar cap */
        nr = 4 * ns - jr; k = 0;
        *zn = -(3 * ns * ns - nr * nr); *zd = 3 * ns * ns;
    } else {                       /* equatorial belt */
        nr = ns; k = (jr - ns) & 1;
        *zn = 2 * (2 * ns - jr); *zd = 3 * ns;
    }
    int64_t num = P[f] * nr + ix - iy + 1 + k;     /* always even */
    int64_t jp = num / 2;
    if (jp > 4 * nr) jp -= 4 * nr;
    if (jp < 1) jp += 4 * nr;
    *m = 2 * jp - k - 1;
    *nr_out = nr;
}

/* sin and cos of phi = m*pi/(4*nr): exact integer octant reduction, then fixed Taylor
 * polynomials in Horner form with separate multiply and add (contract C2). */
void orc_sincos_frac(int64_t m, int64_t nr, double *sinphi, double *cosphi)
{
    const int64_t quad = m / (2 * nr);
    int64_t mr = m % (2 * nr);
    int reflect = 0;
    if (mr > nr) { mr = 2 * nr - mr; reflect = 1; }
    const double beta = (ORC_PI * (double)mr) / (double)(4 * nr);   /* in [0, pi/4] */
    const double u = beta * beta;
    /* sin(beta) = beta + (beta*u)*p(u),  p = -1/3! + u/5! - u^2/7! + ... - u^7/17! */
    double p = 1.0 / 355687428096000.0;           /* 1/17! */
    p = p * u + (-1.0 / 1307674368000.0);         /* 1/15! */
    p = p * u + (1.0 / 6227020800.0);             /* 1/13! */
    p = p * u + (-1.0 / 39916800.0);              /* 1/11! */
    p = p * u + (1.0 / 362880.0);                 /* 1/9!  */
    p = p * u + (-1.0 / 5040.0);                  /* 1/7!  */
    p = p * u + (1.0 / 120.0);                    /* 1/5!  */
    p = p * u + (-1.0 / 6.0);                     /* 1/3!  */
    const double sb = beta + (beta * u) * p;
    /* cos(beta) = 1 - u*(1/2 - u*q(u)),  q = 1/4! - u/6! + u^2/8! - ... + u^7/18! */
    double q = -1.0 / 6402373705728000.0;         /* 1/18! */
    q = q * u + (1.0 / 20922789888000.0);         /* 1/16! */
    q = q * u + (-1.0 / 87178291200.0);           /* 1/14! */
    q = q * u + (1.0 / 479001600.0);              /* 1/12! */
    q = q * u + (-1.0 / 3628800.0);               /* 1/10! */
    q = q * u + (1.0 / 40320.0);                  /* 1/8!  */
    q = q * u + (-1.0 / 720.0);                   /* 1/6!  */
    q = q * u + (1.0 / 24.0);                     /* 1/4!  */
    const double cb = 1.0 - u * (0.5 - u * q);
    const double sa = reflect ? cb : sb;          /* angle inside the quadrant */
    const double ca = reflect ? sb : cb;
    switch (quad) {
        case 0: *cosphi = ca;  *sinphi = sa;  break;
        case 1: *cosphi = -sa; *sinphi = ca;  break;
        case 2: *cosphi = -ca; *sinphi = -sa; break;
        default: *cosphi = sa; *sinphi = -ca; break;
    }
}

void orc_pix2vec(int level, uint64_t pix, double d[3])
{
    int64_t zn, zd, m, nr;
    orc_pix2ring(level, pix, &zn, &zd, &m, &nr);
    const double z = (double)zn / (double)zd;
    const double s = sqrt((1.0 - z) * (1.0 + z));
    double sp, cp;
    orc_sincos_frac(m, nr, &sp, &cp);
    d[0] = s * cp;
    d[1] = s * sp;
    d[2] = z;
}

/* O2. split radius of level l in cell units: Omega_l r^2 = dx^2/Phi  =>  r = sqrt(3/(pi Phi)) 2^l */
double orc_rsplit(double Phi, int level, int Lmax)
{
    if (level >= Lmax) return INFINITY;
    const double c = sqrt(3.0 / (ORC_PI * Phi));
    return ldexp(c, level);
}

/* ------------------------------------------------------------------------------------------
 * O4. opacity table kappa[cell*nb + v] = sum_S sigma_Sv n_S, rounded to the field dtype.
 * ------------------------------------------------------------------------------------------ */
static double n_He_of(double nH, double Yp) { return nH * Yp / (4.0 * (1.0 - Yp)); }

void orc_opacity(const orc_params *p, int nb, const double *nH, const double *xHI, const double *xHeI,
                 const double *xHeII, const double *sHI, const double *sHeI, const double *sHeII,
                 double *kappa)
{
    const int64_t nc = (int64_t)p->N * p->N * p->N;
    for (int64_t c = 0; c < nc; ++c) {
        const double nHe = n_He_of(nH[c], p->Yp);
        const double nHI = nH[c] * xHI[c], nHeI = nHe * xHeI[c], nHeII = nHe * xHeII[c];
        for (int v = 0; v < nb; ++v) {
            double k = (sHI[v] * nHI + sHeI[v] * nHeI) + sHeII[v] * nHeII;
            if (p->field_dtype == 0) k = (double)(float)k;
            kappa[c * nb + v] = k;
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * O3. the ray tracer
 * ------------------------------------------------------------------------------------------ */
typedef struct { int32_t src, level; uint64_t pix; double r0; double tau[ORC_MAXNB]; } ray_rec;

static uint64_t mix64(uint64_t x)      /* splitmix64 finaliser (public-domain constant set) */
{
    x ^= x >> 30; x *= 0xbf58476d1ce4e5b9ull;
    x ^= x >> 27; x *= 0x94d049bb133111ebull;
    x ^= x >> 31;
    return x;
}
static uint64_t ray_key(int32_t src, int32_t level, uint64_t pix)
{
    return ((uint64_t)(uint32_t)src << 40) | ((uint64_t)level << 32) | pix;
}

/* blocked: NULL, or [nsrc][12 4^l0] bytes, non-zero = that root ray is blocked (anisotropic emission, PAPER.md:88:
 * "assigning the mean S_nu per ray to a fraction f_esc of the rays, while completely blocking ... the remaining rays").
 * A blocked root ray does not exist: no packet, no segments, not in emitted. */
/* Optically thin inner region (readings G33-G37), active when p->thin_tau > 0:
 *  Rstart[s] (grid units; NULL = all 0): radius found by the PREVIOUS trace.  Where it is > 0, (iii) every cell whose
 *  centre lies within Rstart of the source receives S_nu kappa_nu V / (4 pi r^2) absorbed photons/s (Eq. 1 for small
 *  tau, dilution 4 pi r^2; r^2 not below (d/2)^2), and (iv) the rays start at r = Rstart with tau = 0, at the level
 *  they would have there (r_split(l-1) <= Rstart < r_split(l)).
 *  Rnext[s] (may be NULL): (ii) the minimum over this trace's rays of the radius up to which tau (softest bin) stays
 *  below thin_tau: the START radius of the segment in which tau reaches thin_tau, or the radius at which a ray ends
 *  (leaves the box / is depleted) with tau still below it; 0 if the source traced no ray. */
int orc_trace_thin(const orc_params *p, int nb, const double *kappa, int nsrc, const double *pos_cm,
                   const double *Ndot, const double *binfrac, const uint8_t *blocked, const double *Rstart,
                   double *Rnext, double *A, orc_stats *st, orc_raylog *log)
{
    const int N = p->N;
    const double dx = p->box_cm / (double)N;
    const int64_t nc = (int64_t)N * N * N;
    memset(st, 0, sizeof(*st));
    memset(A, 0, sizeof(double) * (size_t)nc * nb);
    if (log) { log->n_rays = 0; log->n_cells = 0; }

    size_t cap = 1024, top = 0;
    ray_rec *stack = (ray_rec *)malloc(cap * sizeof(ray_rec));
    if (!stack) return -2;

    for (int s = 0; s < nsrc; ++s) {
        double g[3];
        for (int a = 0; a < 3; ++a) g[a] = pos_cm[3 * s + a] / dx;      /* grid units */
        /* root rays: all pixels of level l0, r = 0, tau = 0 */
        const uint64_t npix0 = 12ull << (2 * p->l0);
        uint64_t nopen = npix0;
        if (blocked) for (uint64_t k = 0; k < npix0; ++k) if (blocked[(uint64_t)s * npix0 + k]) --nopen;
        for (int v = 0; v < nb; ++v) st->emitted[v] += (Ndot[s] * binfrac[s * nb + v]) / (double)npix0 * (double)nopen;
        const int thin = p->thin_tau > 0.0;
        const double R0 = (thin && Rstart) ? Rstart[s] : 0.0;
        double Rmin = INFINITY;
        int lroot = p->l0;
        if (R0 > 0.0) {
            /* (iv) the level rays have at radius R0 */
            while (lroot < p->Lmax && orc_rsplit(p->Phi, lroot, p->Lmax) <= R0) ++lroot;
            /* (iii) cells whose centre is within R0: thin-limit absorption, no rays */
            const double R2 = R0 * R0;
            for (int iz = 0; iz < N; ++iz) for (int iy = 0; iy < N; ++iy) for (int ix = 0; ix < N; ++ix) {
                const double ex = ((double)ix + 0.5) - g[0], ey = ((double)iy + 0.5) - g[1], ez = ((double)iz + 0.5) - g[2];
                const double d2 = (ex * ex + ey * ey) + ez * ez;
                if (!(d2 <= R2)) continue;
                const double r2 = d2 < 0.25 ? 0.25 : d2;
                const int64_t c = ((int64_t)iz * N + iy) * N + ix;
                for (int v = 0; v < nb; ++v) {
                    const double a_v = (Ndot[s] * binfrac[s * nb + v]) / (double)npix0 * (double)nopen
                                       * (kappa[c * nb + v] * dx) / (4.0 * ORC_PI * r2);
                    A[c * nb + v] += a_v; st->absorbed[v] += a_v;
                }
            }
        }
        const uint64_t npixr = 12ull << (2 * lroot);
        for (uint64_t k = npixr; k-- > 0;) {
            if (blocked && blocked[(uint64_t)s * npix0 + (k >> (2 * (lroot - p->l0)))]) continue;   /* blocked level-l0 ancestor */
            if (top == cap) { cap *= 2; stack = (ray_rec *)realloc(stack, cap * sizeof(ray_rec)); if (!stack) return -2; }
            ray_rec *r = &stack[top++];
            r->src = s; r->level = lroot; r->pix = k; r->r0 = R0;
            for (int v = 0; v < nb; ++v) r->tau[v] = 0.0;
        }
        while (top > 0) {
            if (top > st->max_stack) st->max_stack = top;
            ray_rec ray = stack[--top];
            const int l = ray.level;
            double d[3], S[ORC_MAXNB], tau[ORC_MAXNB];
            orc_pix2vec(l, ray.pix, d);
            const double npix = (double)(12ull << (2 * l));
            for (int v = 0; v < nb; ++v) { S[v] = (Ndot[s] * binfrac[s * nb + v]) / npix; tau[v] = ray.tau[v]; }
            const double rs = orc_rsplit(p->Phi, l, p->Lmax);
            double r = ray.r0;
            st->rays++; st->rays_level[l]++;
            uint64_t h = mix64(ray_key(s, l, ray.pix));
            int64_t lr = -1;
            if (log) {
                if (log->n_rays >= log->cap_rays) { free(stack); return -5; }
                lr = log->n_rays++;
                log->src[lr] = s; log->level[lr] = l; log->pix[lr] = (int64_t)ray.pix;
                log->first[lr] = log->n_cells; log->count[lr] = 0;
            }
            /* step 2: starting cell */
            int i[3]; int inside = 1;
            for (int a = 0; a < 3; ++a) {
                const double x = g[a] + r * d[a];
                double fl = floor(x);
                if (x == fl && d[a] < 0.0) fl -= 1.0;
                if (fl < 0.0 || fl >= (double)N) { inside = 0; i[a] = -1; } else i[a] = (int)fl;
            }
            int end;
            if (!inside) {
                for (int v = 0; v < nb; ++v) st->escaped[v] += S[v] * exp(-tau[v]);
                end = ORC_END_ESCAPED;
            } else {
                for (;;) {
                    /* step 3: distance to the next X, Y or Z boundary */
                    double t[3];
                    for (int a = 0; a < 3; ++a) {
                        if (d[a] != 0.0) {
                            const double b = (double)(i[a] + (d[a] > 0.0 ? 1 : 0));
                            t[a] = (b - g[a]) / d[a];
                        } else t[a] = INFINITY;
                    }
                    int ax = 0; double tmin = t[0];
                    if (t[1] < tmin) { tmin = t[1]; ax = 1; }
                    if (t[2] < tmin) { tmin = t[2]; ax = 2; }
                    int split = 0; double r_out = tmin;
                    if (rs <= tmin) { r_out = rs; split = 1; }
                    double ds = r_out - r; if (ds < 0.0) ds = 0.0;
                    /* step 4: deposit (Eq. 1; reading G13: current rate S e^-tau) */
                    const int64_t c = ((int64_t)i[2] * N + i[1]) * N + i[0];
                    const double dl = ds * dx;
                    /* geometric correction (Eq. 2-3; readings G25-G29).  D_edge: distance from the
                     * midpoint of the segment to the nearest of the six cell faces; L_pix: width of the pixel at the
                     * midpoint radius, r_mid sqrt(Omega_l); f_c = 1/2 + D_edge/L_pix if D_edge < L_pix/2, else 1. */
                    double fc = 1.0; int64_t cn = -1;
                    if (p->geom_corr) {
                        const double rmid = 0.5 * (r + r_out);
                        const double Lpix = rmid * ldexp(sqrt(ORC_PI / 3.0), -l);     /* sqrt(4 pi / (12 4^l)) = sqrt(pi/3) / 2^l */
                        double D = INFINITY; int nax = 0, nside = 0;
                        for (int a = 0; a < 3; ++a) {            /* faces in the order x-, x+, y-, y+, z-, z+; first minimum wins */
                            const double m = g[a] + rmid * d[a];
                            const double u = m - (double)i[a];
                            const double hi = 1.0 - u;
                            if (u < D) { D = u; nax = a; nside = -1; }
                            if (hi < D) { D = hi; nax = a; nside = +1; }
                        }
                        if (D < 0.0) D = 0.0;                    /* (rounding can put the midpoint a hair outside) */
                        if (2.0 * D < Lpix) {
                            fc = 0.5 + D / Lpix;
                            if (p->geom_corr == 3) fc = fc * fc;    /* Wise & Abel (2011) form */
                            int j[3] = {i[0], i[1], i[2]};
                            j[nax] += nside;
                            if (j[nax] >= 0 && j[nax] < N) cn = ((int64_t)j[2] * N + j[1]) * N + j[0];
                        }
                    }
                    for (int v = 0; v < nb; ++v) {
                        const double dtau = kappa[c * nb + v] * dl;
                        const double a_v = S[v] * exp(-tau[v]) * (-expm1(-dtau));
                        if (fc == 1.0) { A[c * nb + v] += a_v; st->absorbed[v] += a_v; }
                        else {
                            const double in = fc * a_v, off = a_v - in;          /* in + off = a_v */
                            A[c * nb + v] += in; st->absorbed[v] += in;
                            if (p->geom_corr == 2) {               /* Eq. 3: what f_c removed goes to the nearest adjacent cell */
                                A[(cn >= 0 ? cn : c) * nb + v] += off; st->absorbed[v] += off;
                            }
                        }
                        if (v == 0 && thin && tau[0] < p->thin_tau && tau[0] + dtau >= p->thin_tau && r < Rmin) Rmin = r;   /* (ii) */
                        tau[v] = tau[v] + dtau;
                    }
                    st->segments++;
                    h = mix64(h ^ (uint64_t)c);
                    if (log) {
                        if (log->n_cells >= log->cap_cells) { free(stack); return -5; }
                        log->cells[log->n_cells] = (int32_t)c; log->ds[log->n_cells] = ds;
                        log->n_cells++; log->count[lr]++;
                    }
                    r = r_out;
                    /* step 5: termination on optical depth (reading G7) */
                    double taumin = tau[0];
                    for (int v = 1; v < nb; ++v) if (tau[v] < taumin) taumin = tau[v];
                    if (taumin >= p->tau_term) {
                        for (int v = 0; v < nb; ++v) {
                            const double rem = S[v] * exp(-tau[v]);
                            A[c * nb + v] += rem; st->absorbed[v] += rem;
                        }
                        end = ORC_END_DEPLETED; break;
                    }
                    /* step 6 */
                    if (split) {
                        for (int j = 3; j >= 0; --j) {
                            if (top == cap) { cap *= 2; stack = (ray_rec *)realloc(stack, cap * sizeof(ray_rec)); if (!stack) return -2; }
                            ray_rec *ch = &stack[top++];
                            ch->src = s; ch->level = l + 1; ch->pix = 4 * ray.pix + (uint64_t)j; ch->r0 = r;
                            for (int v = 0; v < nb; ++v) ch->tau[v] = tau[v];
                        }
                        st->splits[l]++;
                        end = ORC_END_SPLIT; break;
                    }
                    i[ax] += (d[ax] > 0.0) ? 1 : -1;
                    if (i[ax] < 0 || i[ax] >= N) {
                        for (int v = 0; v < nb; ++v) st->escaped[v] += S[v] * exp(-tau[v]);
                        end = ORC_END_ESCAPED; break;
                    }
                }
            }
            if (thin && end != ORC_END_SPLIT && tau[0] < p->thin_tau && r < Rmin) Rmin = r;      /* (ii): ended still thin */
            st->ends[end]++;
            h = mix64(h ^ (0xE0ull + (uint64_t)end));
            st->digest += h;
            if (log) { log->end[lr] = end; log->r_end[lr] = r; }
        }
        if (Rnext) Rnext[s] = (thin && Rmin < INFINITY) ? Rmin : 0.0;
    }
    free(stack);
    return 0;
}

int orc_trace_masked(const orc_params *p, int nb, const double *kappa, int nsrc, const double *pos_cm,
                     const double *Ndot, const double *binfrac, const uint8_t *blocked, double *A, orc_stats *st,
                     orc_raylog *log)
{
    return orc_trace_thin(p, nb, kappa, nsrc, pos_cm, Ndot, binfrac, blocked, NULL, NULL, A, st, log);
}

int orc_trace(const orc_params *p, int nb, const double *kappa, int nsrc, const double *pos_cm,
              const double *Ndot, const double *binfrac, double *A, orc_stats *st, orc_raylog *log)
{
    return orc_trace_masked(p, nb, kappa, nsrc, pos_cm, Ndot, binfrac, NULL, A, st, log);
}

/* ------------------------------------------------------------------------------------------
 * O5. finalise: per-cell photo-ionisation rates and heating (Eq. 1 with n_abs = n_SI;
 * PAPER.md:170).  Species share of a bin: proportional to its opacity (reading G8).
 * ------------------------------------------------------------------------------------------ */
static const double ORC_EV = 1.602176634e-12;      /* erg */
static const double ORC_KB = 1.380649e-16;         /* erg/K */
static const double ORC_ETH[3] = {13.598, 24.587, 54.418};

void orc_finalize(const orc_params *p, int nb, const double *A, const double *nH, const double *xHI,
                  const double *xHeI, const double *xHeII, const double *E_eV, const double *sHI,
                  const double *sHeI, const double *sHeII, double *Gamma /*[3][nc]*/,
                  double *heat /*[3][nc]*/, double *heat_total /*[nc]*/)
{
    const int64_t nc = (int64_t)p->N * p->N * p->N;
    const double dx = p->box_cm / (double)p->N;
    const double V = dx * dx * dx;
    for (int64_t c = 0; c < nc; ++c) {
        const double nHe = n_He_of(nH[c], p->Yp);
        const double n[3] = {nH[c] * xHI[c], nHe * xHeI[c], nHe * xHeII[c]};
        double G[3] = {0, 0, 0}, H[3] = {0, 0, 0};
        for (int v = 0; v < nb; ++v) {
            const double sig[3] = {sHI[v], sHeI[v], sHeII[v]};
            const double kp = (sig[0] * n[0] + sig[1] * n[1]) + sig[2] * n[2];
            if (!(kp > 0.0)) continue;
            const double w = A[c * nb + v] / (V * kp);
            for (int S = 0; S < 3; ++S) {
                G[S] += w * sig[S];
                if (E_eV[v] > ORC_ETH[S]) H[S] += w * sig[S] * ((E_eV[v] - ORC_ETH[S]) * ORC_EV);
            }
        }
        for (int S = 0; S < 3; ++S) { Gamma[S * nc + c] = G[S]; heat[S * nc + c] = H[S]; }
        heat_total[c] = (H[0] * n[0] + H[1] * n[1]) + H[2] * n[2];
    }
}

/* ------------------------------------------------------------------------------------------
 * Rate coefficients (reading G11): Hui & Gnedin (1997)-type fits for recombination and
 * collisional ionisation, Cen (1992)-type excitation / bremsstrahlung cooling.
 * Only alpha_B(HII, 1e4 K) = 2.59e-13 is pinned by the paper.
 * out: 0 aHII 1 aHeII 2 aHeIII 3 cHI 4 cHeI 5 cHeII   [cm^3/s]
 *      6 rcHII 7 rcHeII 8 rcHeIII  (recombination cooling, erg cm^3/s, per n_e n_ion)
 *      9 ciHI 10 ciHeI 11 ciHeII   (coll. ionisation cooling, per n_e n_neutral)
 *      12 ceHI 13 ceHeII           (coll. excitation cooling, per n_e n_X)
 *      14 brems                    (per n_e (n_HII + n_HeII + 4 n_HeIII))
 * ------------------------------------------------------------------------------------------ */
void orc_rate_coeffs(double T, int caseB, int coll_ion, double out[15])
{
    const double lH = 2.0 * 157807.0 / T, lHe1 = 2.0 * 285335.0 / T, lHe2 = 2.0 * 631515.0 / T;
    double aHII, aHeII, aHeIII, rcHII, rcHeIII;
    if (caseB) {
        aHII = 2.753e-14 * pow(lH, 1.5) / pow(1.0 + pow(lH / 2.74, 0.407), 2.242);
        aHeII = 1.26e-14 * pow(lHe1, 0.75);
        aHeIII = 2.0 * 2.753e-14 * pow(lHe2, 1.5) / pow(1.0 + pow(lHe2 / 2.74, 0.407), 2.242);
        rcHII = 3.435e-30 * T * pow(lH, 1.97) / pow(1.0 + pow(lH / 2.25, 0.376), 3.72);
        rcHeIII = 8.0 * 3.435e-30 * T * pow(lHe2, 1.97) / pow(1.0 + pow(lHe2 / 2.25, 0.376), 3.72);
    } else {
        aHII = 1.269e-13 * pow(lH, 1.503) / pow(1.0 + pow(lH / 0.522, 0.47), 1.923);
        aHeII = 3.0e-14 * pow(lHe1, 0.654);
        aHeIII = 2.0 * 1.269e-13 * pow(lHe2, 1.503) / pow(1.0 + pow(lHe2 / 0.522, 0.47), 1.923);
        rcHII = 1.778e-29 * T * pow(lH, 1.965) / pow(1.0 + pow(lH / 0.541, 0.502), 2.697);
        rcHeIII = 8.0 * 1.778e-29 * T * pow(lHe2, 1.965) / pow(1.0 + pow(lHe2 / 0.541, 0.502), 2.697);
    }
    /* dielectronic recombination of He II */
    const double ad = 1.9e-3 * pow(T, -1.5) * exp(-470000.0 / T) * (1.0 + 0.3 * exp(-94000.0 / T));
    out[0] = aHII; out[1] = aHeII + ad; out[2] = aHeIII;
    double cHI = 0, cHeI = 0, cHeII = 0;
    if (coll_ion) {
        cHI = 21.11 * pow(T, -1.5) * exp(-lH / 2.0) * pow(lH, -1.089) / pow(1.0 + pow(lH / 0.354, 0.874), 1.101);
        cHeI = 32.38 * pow(T, -1.5) * exp(-lHe1 / 2.0) * pow(lHe1, -1.146) / pow(1.0 + pow(lHe1 / 0.416, 0.987), 1.056);
        cHeII = 19.95 * pow(T, -1.5) * exp(-lHe2 / 2.0) * pow(lHe2, -1.089) / pow(1.0 + pow(lHe2 / 0.553, 0.735), 1.275);
    }
    out[3] = cHI; out[4] = cHeI; out[5] = cHeII;
    out[6] = rcHII; out[7] = ORC_KB * T * aHeII + 6.54e-11 * ad; out[8] = rcHeIII;
    out[9] = 2.18e-11 * cHI; out[10] = 3.94e-11 * cHeI; out[11] = 8.72e-11 * cHeII;
    const double f5 = 1.0 / (1.0 + sqrt(T / 1.0e5));
    out[12] = 7.5e-19 * exp(-118348.0 / T) * f5;
    out[13] = 5.54e-17 * pow(T, -0.397) * exp(-473638.0 / T) * f5;
    const double lg = log10(T);
    const double gff = 1.1 + 0.34 * exp(-(5.5 - lg) * (5.5 - lg) / 3.0);
    out[14] = 1.42e-27 * gff * sqrt(T);
}

/* ------------------------------------------------------------------------------------------
 * O6. chemistry / thermal update of one cell over dt.
 * state x = {xHI, xHeI, xHeII}, T.  G = photo-ionisation rates per absorber [1/s],
 * H = heating per absorber [erg/s] - held fixed during the call.
 * Returns the number of sub-cycles taken.
 * ------------------------------------------------------------------------------------------ */
static double clampd(double v, double lo, double hi) { return v < lo ? lo : (v > hi ? hi : v); }

int orc_chem_cell(const orc_params *p, double nH, double x[3], double *T, const double G[3],
                  const double H[3], double dt)
{
    const double nHe = n_He_of(nH, p->Yp);
    double t = 0.0;
    int k = 0;
    double co[15];
    if (p->isothermal) orc_rate_coeffs(*T, p->caseB, p->coll_ion, co);
    while (t < dt && k < p->max_subcycles) {
        const double xHII = 1.0 - x[0];
        double xHeIII = 1.0 - x[1] - x[2]; if (xHeIII < 0.0) xHeIII = 0.0;
        const double ne = nH * xHII + nHe * (x[2] + 2.0 * xHeIII);
        if (!p->isothermal) orc_rate_coeffs(*T, p->caseB, p->coll_ion, co);
        /* Eq. 4 in the form of Eq. 5, per species, in fractions */
        const double C0 = G[0] + co[3] * ne, D0 = co[0] * ne * xHII;
        const double C1 = G[1] + co[4] * ne, D1 = co[1] * ne * x[2];
        const double C2 = (G[2] + co[5] * ne) + co[1] * ne;
        const double D2 = (G[1] + co[4] * ne) * x[1] + co[2] * ne * xHeIII;
        const double xdot0 = D0 - C0 * x[0];
        double dts = dt - t;
        const int last = (k == p->max_subcycles - 1);
        double heat = 0.0, cool = 0.0, E = 0.0;
        if (!p->isothermal) {
            const double nHI = nH * x[0], nHeI = nHe * x[1], nHeII = nHe * x[2];
            const double nHII = nH * xHII, nHeIII = nHe * xHeIII;
            heat = (H[0] * nHI + H[1] * nHeI) + H[2] * nHeII;
            cool = ne * (co[6] * nHII + co[7] * nHeII + co[8] * nHeIII
                         + co[9] * nHI + co[10] * nHeI + co[11] * nHeII
                         + co[12] * nHI + co[13] * nHeII
                         + co[14] * (nHII + nHeII + 4.0 * nHeIII));
            E = 1.5 * ORC_KB * (*T) * (nH + nHe + ne);
        }
        if (!last) {
            if (xdot0 != 0.0) { const double l = p->eps_sub * x[0] / fabs(xdot0); if (l < dts) dts = l; }
            if (!p->isothermal && heat - cool != 0.0) {
                const double l = p->eps_sub * E / fabs(heat - cool); if (l < dts) dts = l;
            }
        }
        /* backward difference (Eq. 5): n <- (n + D dt)/(1 + C dt), Jacobi order (reading G16) */
        const double y0 = (x[0] + D0 * dts) / (1.0 + C0 * dts);
        const double y1 = (x[1] + D1 * dts) / (1.0 + C1 * dts);
        const double y2 = (x[2] + D2 * dts) / (1.0 + C2 * dts);
        x[0] = clampd(y0, p->x_floor, 1.0);
        x[1] = clampd(y1, p->x_floor, 1.0);
        x[2] = clampd(y2, 0.0, 1.0);
        if (x[1] + x[2] > 1.0) { const double sum = x[1] + x[2]; x[1] = x[1] / sum; x[2] = x[2] / sum; }
        if (!p->isothermal) {
            const double En = (E + heat * dts) / (1.0 + (cool / E) * dts);
            const double xHII_n = 1.0 - x[0];
            double xHeIII_n = 1.0 - x[1] - x[2]; if (xHeIII_n < 0.0) xHeIII_n = 0.0;
            const double ne_n = nH * xHII_n + nHe * (x[2] + 2.0 * xHeIII_n);
            double Tn = En / (1.5 * ORC_KB * (nH + nHe + ne_n));
            if (Tn < 1.0) Tn = 1.0;
            *T = Tn;
        }
        t = (dts >= dt - t) ? dt : t + dts;
        ++k;
    }
    return k;
}

/* whole grid; fields updated in place (fp64 here; the caller rounds to f32 if the run is f32) */
int64_t orc_chemistry(const orc_params *p, const double *nH, double *xHI, double *xHeI, double *xHeII,
                      double *T, const double *Gamma, const double *heat, double dt, int32_t *subcycles)
{
    const int64_t nc = (int64_t)p->N * p->N * p->N;
    int64_t total = 0;
    for (int64_t c = 0; c < nc; ++c) {
        double x[3] = {xHI[c], xHeI[c], xHeII[c]};
        double Tc = T[c];
        const double G[3] = {Gamma[c], Gamma[nc + c], Gamma[2 * nc + c]};
        const double H[3] = {heat[c], heat[nc + c], heat[2 * nc + c]};
        const int k = orc_chem_cell(p, nH[c], x, &Tc, G, H, dt);
        if (p->field_dtype == 0) {
            xHI[c] = (double)(float)x[0]; xHeI[c] = (double)(float)x[1]; xHeII[c] = (double)(float)x[2];
            T[c] = (double)(float)Tc;
        } else { xHI[c] = x[0]; xHeI[c] = x[1]; xHeII[c] = x[2]; T[c] = Tc; }
        if (subcycles) subcycles[c] = k;
        total += k;
    }
    return total;
}

/* ------------------------------------------------------------------------------------------
 * Radiative-transfer time step (readings G30-G31).  Per cell, with the rates of the
 * last trace and the current fields: dn_HI/dt = n_H (D - C x_HI) with Eq. 4's D = alpha_HII n_e x_HII,
 * C = Gamma_HI + C_HI n_e.  scheme 1 (:182-190): dt_n = eps n_HI / |dn_HI/dt| over the cells with
 * tau = n_HI sigma_1 d > 0.5; scheme 2 (:192-204): dt_I = eps / (sigma_1 d |dn_HI/dt|) over all cells.  Returns the
 * minimum (+inf if no cell qualifies or nothing changes); *n_used = cells that entered the minimum.
 * ------------------------------------------------------------------------------------------ */
double orc_suggest_dt(const orc_params *p, int scheme, double eps, double sigma1, const double *nH, const double *xHI,
                      const double *xHeI, const double *xHeII, const double *T, const double *GammaHI, int64_t *n_used)
{
    const int64_t nc = (int64_t)p->N * p->N * p->N;
    const double d = p->box_cm / (double)p->N;
    double best = INFINITY;
    int64_t used = 0;
    for (int64_t c = 0; c < nc; ++c) {
        const double nHe = n_He_of(nH[c], p->Yp);
        const double xHII = 1.0 - xHI[c];
        double xHeIII = 1.0 - xHeI[c] - xHeII[c]; if (xHeIII < 0.0) xHeIII = 0.0;
        const double ne = nH[c] * xHII + nHe * (xHeII[c] + 2.0 * xHeIII);
        double co[15];
        orc_rate_coeffs(T[c], p->caseB, p->coll_ion, co);
        const double C0 = GammaHI[c] + co[3] * ne, D0 = co[0] * ne * xHII;
        const double nHI = nH[c] * xHI[c];
        const double ndot = fabs(nH[c] * (D0 - C0 * xHI[c]));
        if (ndot == 0.0) continue;
        double dt;
        if (scheme == 1) {
            const double tau = (nHI * sigma1) * d;
            if (!(tau > 0.5)) continue;
            dt = eps * nHI / ndot;
        } else dt = eps / ((sigma1 * d) * ndot);
        ++used;
        if (dt < best) best = dt;
    }
    if (n_used) *n_used = used;
    return best;
}

int orc_sizeof_params(void) { return (int)sizeof(orc_params); }
int orc_sizeof_stats(void) { return (int)sizeof(orc_stats); }
