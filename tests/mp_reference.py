"""The finite sum of DESIGN.md section 1 written out term by term with mpmath at a chosen number of
digits, on the oracle's own nodes and weights (massive lines only).  Independent of the CUDA path.

Used (a) to pin the oracle's parity variant: its own rounding error must be << 1e-11 (reading G18), and
(b) as the reference where no fixed-width arithmetic can evaluate the plain sum: for |x| below ~1e-30 the
+-z terms, each O(sqrt|x y|), cancel to O(|x|), a loss of 2 sqrt(y/|x|) that exceeds even binary128.
"""
import mpmath as mp


def finite_sum(oracle, P, x, rad_nodes, rad_weights, n_rad, z, wz, digits=60):
    """c0 sum_i wy_i y_i D1(y_i) sum_j w'_j [D2(u_ij) - D2(y_i)] in the combined form of eq. (20)
    (PAPER.md:198-203), u_ij = y_i + d_ij, d_ij = x - 2 sqrt(x) sqrt(y_i) z_j (eq. (10))."""
    x = complex(x)
    _, ys, wys = oracle.contour_nodes(P, x, rad_nodes, rad_weights, n_rad, len(z))
    assert P.line_k.kind == 0 and P.line_pk.kind == 0, "massive lines only"
    with mp.workdps(digits):
        m1 = mp.mpc(P.line_k.m2_re, P.line_k.m2_im)
        m2 = mp.mpc(P.line_pk.m2_re, P.line_pk.m2_im)
        xm = mp.mpc(x.real, x.imag)
        sx, g = mp.sqrt(xm), mp.mpc(0)
        for yi, wyi in zip(ys, wys):
            y = mp.mpc(yi.real, yi.imag)
            B, c, S = 2 * sx * mp.sqrt(y), y + m2, mp.mpc(0)
            for zj, wj in zip(z, wz):
                d = xm - B * mp.mpf(float(zj))
                S += mp.mpf(float(wj)) * (-d / ((c + d) * c)) / (y + m1)
            g += mp.mpc(wyi.real, wyi.imag) * y * S
        return complex(mp.mpf(P.prefactor) * g)
