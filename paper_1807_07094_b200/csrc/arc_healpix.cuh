// arc_healpix.cuh -- device HEALPix nested pix2vec and child generation.
// Direction of pixel p at level l (Gorski et al. 2005, cited PAPER.md:45, 88), following DESIGN.md
// contract C1-C2: integer ring coordinates, z from ONE fp64 division of exact integers, sin/cos of
// phi = m*pi/(4*nr) by exact integer octant reduction and fixed Taylor polynomials evaluated with
// separate IEEE multiplies and adds (no FMA), so that the result is bit-identical on any IEEE machine.
// Children of p at level l+1 are 4p..4p+3 ("breaks this area into four sub-areas").
#pragma once
#include <stdint.h>

__device__ __forceinline__ uint32_t arc_compact_even_bits(uint32_t v)
{
    v &= 0x55555555u;
    v = (v | (v >> 1)) & 0x33333333u;
    v = (v | (v >> 2)) & 0x0F0F0F0Fu;
    v = (v | (v >> 4)) & 0x00FF00FFu;
    v = (v | (v >> 8)) & 0x0000FFFFu;
    return v;
}

__device__ __forceinline__ double arc_mul(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ double arc_add(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ double arc_sub(double a, double b) { return __dsub_rn(a, b); }

// sin, cos of beta in [0, pi/4]; Horner, multiply and add kept separate (contract C2)
__device__ __forceinline__ void arc_sincos_octant(double beta, double &sb, double &cb)
{
    const double u = arc_mul(beta, beta);
    double p = 1.0 / 355687428096000.0;
    p = arc_add(arc_mul(p, u), -1.0 / 1307674368000.0);
    p = arc_add(arc_mul(p, u), 1.0 / 6227020800.0);
    p = arc_add(arc_mul(p, u), -1.0 / 39916800.0);
    p = arc_add(arc_mul(p, u), 1.0 / 362880.0);
    p = arc_add(arc_mul(p, u), -1.0 / 5040.0);
    p = arc_add(arc_mul(p, u), 1.0 / 120.0);
    p = arc_add(arc_mul(p, u), -1.0 / 6.0);
    sb = arc_add(beta, arc_mul(arc_mul(beta, u), p));
    double q = -1.0 / 6402373705728000.0;
    q = arc_add(arc_mul(q, u), 1.0 / 20922789888000.0);
    q = arc_add(arc_mul(q, u), -1.0 / 87178291200.0);
    q = arc_add(arc_mul(q, u), 1.0 / 479001600.0);
    q = arc_add(arc_mul(q, u), -1.0 / 3628800.0);
    q = arc_add(arc_mul(q, u), 1.0 / 40320.0);
    q = arc_add(arc_mul(q, u), -1.0 / 720.0);
    q = arc_add(arc_mul(q, u), 1.0 / 24.0);
    cb = arc_sub(1.0, arc_mul(u, arc_sub(0.5, arc_mul(u, q))));
}

__device__ __forceinline__ void arc_pix2vec_dev(int level, uint32_t pix, double &vx, double &vy, double &vz)
{
    const int ns = 1 << level;
    const int face = (int)(pix >> (2 * level));
    const uint32_t q = pix & ((1u << (2 * level)) - 1u);
    const int ix = (int)arc_compact_even_bits(q);
    const int iy = (int)arc_compact_even_bits(q >> 1);
    const int band = face >> 2;                           // 0 north, 1 equatorial, 2 south faces
    const int jr = (band + 2) * ns - ix - iy - 1;         // ring index from the north pole
    int nr, k;
    long long zn, zd;
    if (jr < ns) {                                        // north polar cap
        nr = jr; k = 0;
        zd = 3ll * ns * ns; zn = zd - (long long)nr * nr;
    } else if (jr > 3 * ns) {                             // south polar cap
        nr = 4 * ns - jr; k = 0;
        zd = 3ll * ns * ns; zn = (long long)nr * nr - zd;
    } else {                                              // equatorial belt
        nr = ns; k = (jr - ns) & 1;
        zd = 3ll * ns; zn = 2ll * (2 * ns - jr);
    }
    const int jpl = (band == 1) ? 2 * (face & 3) : 2 * (face & 3) + 1;   // longitude offset of the face
    int jp = (jpl * nr + ix - iy + 1 + k) >> 1;           // numerator is always even
    if (jp > 4 * nr) jp -= 4 * nr;
    if (jp < 1) jp += 4 * nr;
    const int m = 2 * jp - k - 1;                         // phi = m*pi/(4 nr), 0 <= m < 8 nr
    const int quad = m / (2 * nr);
    int mr = m - quad * 2 * nr;
    const bool reflect = mr > nr;
    if (reflect) mr = 2 * nr - mr;
    const double PI = 3.14159265358979323846;
    const double beta = __ddiv_rn(arc_mul(PI, (double)mr), (double)(4 * nr));
    double sb, cb;
    arc_sincos_octant(beta, sb, cb);
    const double sa = reflect ? cb : sb;
    const double ca = reflect ? sb : cb;
    double sp, cp;
    switch (quad) {
        case 0: cp = ca; sp = sa; break;
        case 1: cp = -sa; sp = ca; break;
        case 2: cp = -ca; sp = -sa; break;
        default: cp = sa; sp = -ca; break;
    }
    const double z = __ddiv_rn((double)zn, (double)zd);
    const double s = __dsqrt_rn(arc_mul(arc_sub(1.0, z), arc_add(1.0, z)));
    vx = arc_mul(s, cp);
    vy = arc_mul(s, sp);
    vz = z;
}
