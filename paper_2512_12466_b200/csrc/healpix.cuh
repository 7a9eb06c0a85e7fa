// HEALPix nested pixel centre -> unit vector on the device ("DIR-SPEC").
// Geometry of Gorski et al. 2005 (PAPER.md:613 ref [63]); the paper uses it for the 12 level-0 rays
// and the four children of a split.  Every operation below feeds
// decisions (DEC): integer work is exact, the floating-point sequence is fixed and the file is compiled
// with -fmad=false, so no product-sum is contracted unless fma() is written.
#pragma once
#include <stdint.h>

namespace nyxrt {

// gather the even-position bits of v into the low half
__device__ __forceinline__ uint32_t compact_even_bits(uint32_t v) {
    v &= 0x55555555u;
    v = (v | (v >> 1)) & 0x33333333u;
    v = (v | (v >> 2)) & 0x0f0f0f0fu;
    v = (v | (v >> 4)) & 0x00ff00ffu;
    v = (v | (v >> 8)) & 0x0000ffffu;
    return v;
}

// sin x = x P(x^2), Taylor through x^17; cos x = Q(x^2), Taylor through x^18; Horner, one fma per step.
// Coefficients are +-1/n! rounded once (n! is exact in binary64 up to 18!).
__device__ __forceinline__ double sin_taylor17(double x) {
    const double u = x * x;
    double p = 1.0 / 355687428096000.0;             //  1/17!
    p = fma(p, u, -1.0 / 1307674368000.0);           // -1/15!
    p = fma(p, u, 1.0 / 6227020800.0);               //  1/13!
    p = fma(p, u, -1.0 / 39916800.0);                // -1/11!
    p = fma(p, u, 1.0 / 362880.0);                   //  1/9!
    p = fma(p, u, -1.0 / 5040.0);                    // -1/7!
    p = fma(p, u, 1.0 / 120.0);                      //  1/5!
    p = fma(p, u, -1.0 / 6.0);                       // -1/3!
    p = fma(p, u, 1.0);
    return x * p;
}

__device__ __forceinline__ double cos_taylor18(double x) {
    const double u = x * x;
    double q = -1.0 / 6402373705728000.0;            // -1/18!
    q = fma(q, u, 1.0 / 20922789888000.0);           //  1/16!
    q = fma(q, u, -1.0 / 87178291200.0);             // -1/14!
    q = fma(q, u, 1.0 / 479001600.0);                //  1/12!
    q = fma(q, u, -1.0 / 3628800.0);                 // -1/10!
    q = fma(q, u, 1.0 / 40320.0);                    //  1/8!
    q = fma(q, u, -1.0 / 720.0);                     // -1/6!
    q = fma(q, u, 1.0 / 24.0);                       //  1/4!
    q = fma(q, u, -0.5);                             // -1/2!
    q = fma(q, u, 1.0);
    return q;
}

// level <= 14, pix < 12 * 4^level (fits 32 bits up to level 14)
__device__ __forceinline__ void pix2dir(int level, uint32_t pix, double &dx, double &dy, double &dz) {
    const int ns = 1 << level;
    const uint32_t face = pix >> (2 * level);                    // 0..11
    const uint32_t pf = pix & ((1u << (2 * level)) - 1u);
    const int ix = (int)compact_even_bits(pf);
    const int iy = (int)compact_even_bits(pf >> 1);
    const int row = (int)(face >> 2);                            // 0 north, 1 equatorial, 2 south faces
    const int jr = (row + 2) * ns - ix - iy - 1;                 // ring index, 1 at the north pole
    int nr, k;
    double z, st;
    if (jr < ns) {                                               // north polar cap
        nr = jr; k = 0;
        const double t = (double)(nr * nr) / (double)(3 * ns * ns);
        z = 1.0 - t;
        st = sqrt(t * (2.0 - t));
    } else if (jr > 3 * ns) {                                    // south polar cap
        nr = 4 * ns - jr; k = 0;
        const double t = (double)(nr * nr) / (double)(3 * ns * ns);
        z = t - 1.0;
        st = sqrt(t * (2.0 - t));
    } else {                                                     // equatorial belt
        nr = ns; k = (jr - ns) & 1;
        z = ((double)(2 * ns - jr) * 2.0) / (double)(3 * ns);
        st = sqrt((1.0 - z) * (1.0 + z));
    }
    const int jf = 2 * (int)(face & 3u) + (row == 1 ? 0 : 1);
    int jp = (jf * nr + ix - iy + 1 + k) >> 1;                   // negative only in the belt, where it is even
    if (jp > 4 * nr) jp -= 4 * nr;
    if (jp < 1) jp += 4 * nr;
    const int m = 2 * jp - k - 1;                                // phi = (pi/4) m / nr, 0 <= m < 8 nr
    const int q = m / nr, rem = m - q * nr;
    const int num = (q & 1) ? (nr - rem) : rem;
    const double PI_4 = 0x1.921fb54442d18p-1;
    const double alpha = (PI_4 * (double)num) / (double)nr;      // in [0, pi/4]
    double c = cos_taylor18(alpha), s = sin_taylor17(alpha);
    if (num == nr) { c = 0x1.6a09e667f3bcdp-1; s = c; }          // on a diagonal: cos = sin = sqrt(1/2)
    double cp, sp;
    switch (q) {
        case 0: cp = c;  sp = s;  break;
        case 1: cp = s;  sp = c;  break;
        case 2: cp = -s; sp = c;  break;
        case 3: cp = -c; sp = s;  break;
        case 4: cp = -c; sp = -s; break;
        case 5: cp = -s; sp = -c; break;
        case 6: cp = s;  sp = -c; break;
        default: cp = c; sp = -s; break;
    }
    dx = st * cp;
    dy = st * sp;
    dz = z;
}

}  // namespace nyxrt
