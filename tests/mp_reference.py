"""The finite sum of DESIGN.md section 1 written out term by term with mpmath at a chosen number of
digits, on the oracle's own nodes and weights.  Independent of the CUDA path.

Used (a) to pin the oracle's parity variant: its own rounding error must be << 1e-11 (reading G18), and
(b) as the reference where no fixed-width arithmetic can evaluate the plain sum: for |x| below ~1e-30 the
+-z terms, each O(sqrt|x y|), cancel to O(|x|), a loss of 2 sqrt(y/|x|) that exceeds even binary128.
"""
import mpmath as mp


def _prop(p):
    """The propagator of a line as an mpmath function of its momentum squared (include/gf.h, gf_propagator)."""
    if p.kind == 0:
        m2 = mp.mpc(p.m2_re, p.m2_im)
        return lambda u: 1 / (u + m2)
    M2, a, b = mp.mpf(p.M2), mp.mpf(p.a), mp.mpf(p.b)
    return lambda u: (u + M2) / (u * u + a * u + b)


def finite_sum(oracle, P, x, rad_nodes, rad_weights, n_rad, z, wz, digits=60):
    """c0 sum_i wy_i y_i sum_j w'_j F_sub(x, y_i, z_j) with F_sub = (1 - t^n) F written out as eq. (12),(13) define it
    (PAPER.md:80-87): F itself minus its Taylor polynomial in the external momentum, by plain subtraction at `digits`
    digits.  F = D1(y) D2(u), u = y + d, d = x - 2 sqrt(x) sqrt(y) z (eq. (10),(19)).  With p -> eps p the integrand
    is F(eps) = D1(y) D2(y + eps^2 x - eps 2 sqrt(x) sqrt(y) z), and t^n F is its Taylor polynomial of degree 2n at
    eps = 1 (reading G20; n = 0: F at p = 0, eq. (20)), taken here by numerical differentiation
    (mpmath.taylor), not by any formula of the oracle's."""
    x = complex(x)
    _, ys, wys = oracle.contour_nodes(P, x, rad_nodes, rad_weights, n_rad, len(z))
    n = int(P.taylor_order)
    with mp.workdps(digits + 40 * n):
        D1, D2 = _prop(P.line_k), _prop(P.line_pk)
        xm = mp.mpc(x.real, x.imag)
        sx, g = mp.sqrt(xm), mp.mpc(0)
        for yi, wyi in zip(ys, wys):
            y = mp.mpc(yi.real, yi.imag)
            B, S = 2 * sx * mp.sqrt(y), mp.mpc(0)
            for zj, wj in zip(z, wz):
                zz = mp.mpf(float(zj))
                F = lambda eps: D1(y) * D2(y + eps * eps * xm - eps * B * zz)
                tn = F(0) if n == 0 else mp.fsum(mp.taylor(F, 0, 2 * n))
                S += mp.mpf(float(wj)) * (F(1) - tn)
            g += mp.mpc(wyi.real, wyi.imag) * y * S
        return complex(mp.mpf(P.prefactor) * g)
