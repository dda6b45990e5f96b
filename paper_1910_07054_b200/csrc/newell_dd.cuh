// newell_dd.cuh -- the Newell primitives f (Eq.10) and g (Eq.16)
// in double-double, evaluated for all six tensor components at one lattice point at once.
//
// Components c = 0..5 = xx, yy, zz, xy, xz, yz use ("by permutation of the variables")
//   phi0 = f(x,y,z)  phi1 = f(y,x,z)  phi2 = f(z,x,y)  phi3 = g(x,y,z)  phi4 = g(x,z,y)  phi5 = g(y,z,x)
// Written out, the six share three inverse hyperbolic sines and three arctangents:
//   Lx = asinh(x / sqrt(y^2+z^2))   Tx = atan(y z / (x R))      R = sqrt(x^2+y^2+z^2)
//   Ly = asinh(y / sqrt(x^2+z^2))   Ty = atan(x z / (y R))
//   Lz = asinh(z / sqrt(x^2+y^2))   Tz = atan(x y / (z R))
// A term whose polynomial prefactor vanishes is 0 (the limit; reading A5): Lx is only ever
// multiplied by a factor that vanishes when y = z = 0, Tx by a positive power of x, etc., so
// setting L := 0 / T := 0 where their argument is 0/0 or infinite implements that reading.
// Arguments are taken on |x|,|y|,|z| (principal value of the quotient, reading A6); the caller
// restores signs from the parities of f (even in all) and g (odd, odd, even).
#pragma once
#include "dd.cuh"

namespace hfft {

// phi[0..5] at x, y, z >= 0
DD_D void newell_phi6(dd x, dd y, dd z, dd phi[6]) {
    const dd zero = dd_make(0.0, 0.0);
    dd x2 = dd_sqr(x), y2 = dd_sqr(y), z2 = dd_sqr(z);
    dd xy2 = dd_add(x2, y2), xz2 = dd_add(x2, z2), yz2 = dd_add(y2, z2);
    dd R = dd_sqrt(dd_add(xy2, z2));
    bool x0 = dd_is_zero(x), y0 = dd_is_zero(y), z0 = dd_is_zero(z);

    dd Lx = zero, Ly = zero, Lz = zero, Tx = zero, Ty = zero, Tz = zero;
    if (!x0 && !(y0 && z0)) Lx = dd_asinh_pos(dd_div(x, dd_sqrt(yz2)));
    if (!y0 && !(x0 && z0)) Ly = dd_asinh_pos(dd_div(y, dd_sqrt(xz2)));
    if (!z0 && !(x0 && y0)) Lz = dd_asinh_pos(dd_div(z, dd_sqrt(xy2)));
    if (!x0 && !y0 && !z0) {
        Tx = dd_atan_pos(dd_div(dd_mul(y, z), dd_mul(x, R)));
        Ty = dd_atan_pos(dd_div(dd_mul(x, z), dd_mul(y, R)));
        Tz = dd_atan_pos(dd_div(dd_mul(x, y), dd_mul(z, R)));
    }
    dd xyz = dd_mul(dd_mul(x, y), z);
    const dd sixth = dd_make(DD_TAB_ODDINV[1][0] * 0.5, DD_TAB_ODDINV[1][1] * 0.5);   // 1/6
    const dd third = dd_make(DD_TAB_ODDINV[1][0], DD_TAB_ODDINV[1][1]);               // 1/3
    dd R6 = dd_mul(R, sixth);

    // f(a,b,c) = b/2 (c^2-a^2) asinh(b/sqrt(a^2+c^2)) + c/2 (b^2-a^2) asinh(c/sqrt(a^2+b^2))
    //            - abc atan(bc/(aR)) + (2a^2-b^2-c^2) R/6                              (Eq.10)
    // phi0 = f(x,y,z)
    {
        dd t1 = dd_mul(dd_mul(dd_scale2(y, 0.5), dd_sub(z2, x2)), Ly);
        dd t2 = dd_mul(dd_mul(dd_scale2(z, 0.5), dd_sub(y2, x2)), Lz);
        dd t3 = dd_mul(xyz, Tx);
        dd t4 = dd_mul(dd_sub(dd_scale2(x2, 2.0), yz2), R6);
        phi[0] = dd_add(dd_sub(dd_add(t1, t2), t3), t4);
    }
    // phi1 = f(y,x,z)
    {
        dd t1 = dd_mul(dd_mul(dd_scale2(x, 0.5), dd_sub(z2, y2)), Lx);
        dd t2 = dd_mul(dd_mul(dd_scale2(z, 0.5), dd_sub(x2, y2)), Lz);
        dd t3 = dd_mul(xyz, Ty);
        dd t4 = dd_mul(dd_sub(dd_scale2(y2, 2.0), xz2), R6);
        phi[1] = dd_add(dd_sub(dd_add(t1, t2), t3), t4);
    }
    // phi2 = f(z,x,y)
    {
        dd t1 = dd_mul(dd_mul(dd_scale2(x, 0.5), dd_sub(y2, z2)), Lx);
        dd t2 = dd_mul(dd_mul(dd_scale2(y, 0.5), dd_sub(x2, z2)), Ly);
        dd t3 = dd_mul(xyz, Tz);
        dd t4 = dd_mul(dd_sub(dd_scale2(z2, 2.0), xy2), R6);
        phi[2] = dd_add(dd_sub(dd_add(t1, t2), t3), t4);
    }
    // g(a,b,c) = abc asinh(c/sqrt(a^2+b^2)) + b/6 (3c^2-b^2) asinh(a/sqrt(b^2+c^2))
    //          + a/6 (3c^2-a^2) asinh(b/sqrt(a^2+c^2)) - c^3/6 atan(ab/(cR))
    //          - c b^2/2 atan(ac/(bR)) - c a^2/2 atan(bc/(aR)) - abR/3                  (Eq.16)
    dd x3 = dd_mul(x2, x), y3 = dd_mul(y2, y), z3 = dd_mul(z2, z);
    dd R3 = dd_mul(R, third);
    // phi3 = g(x,y,z)
    {
        dd s = dd_mul(xyz, Lz);
        s = dd_add(s, dd_mul(dd_mul(dd_mul(y, sixth), dd_sub(dd_mul_d(z2, 3.0), y2)), Lx));
        s = dd_add(s, dd_mul(dd_mul(dd_mul(x, sixth), dd_sub(dd_mul_d(z2, 3.0), x2)), Ly));
        s = dd_sub(s, dd_mul(dd_mul(z3, sixth), Tz));
        s = dd_sub(s, dd_mul(dd_scale2(dd_mul(z, y2), 0.5), Ty));
        s = dd_sub(s, dd_mul(dd_scale2(dd_mul(z, x2), 0.5), Tx));
        phi[3] = dd_sub(s, dd_mul(dd_mul(x, y), R3));
    }
    // phi4 = g(x,z,y)
    {
        dd s = dd_mul(xyz, Ly);
        s = dd_add(s, dd_mul(dd_mul(dd_mul(z, sixth), dd_sub(dd_mul_d(y2, 3.0), z2)), Lx));
        s = dd_add(s, dd_mul(dd_mul(dd_mul(x, sixth), dd_sub(dd_mul_d(y2, 3.0), x2)), Lz));
        s = dd_sub(s, dd_mul(dd_mul(y3, sixth), Ty));
        s = dd_sub(s, dd_mul(dd_scale2(dd_mul(y, z2), 0.5), Tz));
        s = dd_sub(s, dd_mul(dd_scale2(dd_mul(y, x2), 0.5), Tx));
        phi[4] = dd_sub(s, dd_mul(dd_mul(x, z), R3));
    }
    // phi5 = g(y,z,x)
    {
        dd s = dd_mul(xyz, Lx);
        s = dd_add(s, dd_mul(dd_mul(dd_mul(z, sixth), dd_sub(dd_mul_d(x2, 3.0), z2)), Ly));
        s = dd_add(s, dd_mul(dd_mul(dd_mul(y, sixth), dd_sub(dd_mul_d(x2, 3.0), y2)), Lz));
        s = dd_sub(s, dd_mul(dd_mul(x3, sixth), Tx));
        s = dd_sub(s, dd_mul(dd_scale2(dd_mul(x, z2), 0.5), Tz));
        s = dd_sub(s, dd_mul(dd_scale2(dd_mul(x, y2), 0.5), Ty));
        phi[5] = dd_sub(s, dd_mul(dd_mul(y, z), R3));
    }
}

}  // namespace hfft
