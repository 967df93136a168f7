"""Closed forms used to pin the oracle.  Independent mathematics: nothing here
calls or restates the oracle's quadrature; all of it is evaluated with mpmath
at 30 digits.

CF1  equal real mass m, c0 = 2/pi: the textbook one-loop bubble, once subtracted at x=0,
       G(x) = 2 - beta ln((beta+1)/(beta-1)),  beta = sqrt(1 + 4 m^2/x)
     (branch cut exactly x <= -4 m^2, the two-particle threshold of PAPER.md:15).
CF2  the paper's worked example, masses^2 +i/2 (k line) and -i/2 (p-k line):
       eq. (18):  1 - pi/(2x) + sqrt(1-x^2) arccos(x) / x
     with w = sqrt(1-x^2), arccos x := -i ln(x + i w) (consistent branches).
CF3  unequal / complex masses a (line k), b (line p-k), Feynman parameter form
       B(x;a,b) = - int_0^1 d alpha  ln(1 + alpha (1-alpha) x / (alpha a + (1-alpha) b));
     a rational line 2 is a sum over its poles, G = sum_r R_r B(x; m1^2, -u_r).
"""
import mpmath as mp

mp.mp.dps = 30


def cf1(x, m2=1.0):
    x = mp.mpc(x)
    if x == 0:
        return mp.mpc(0)
    beta = mp.sqrt(1 + 4 * mp.mpf(m2) / x)
    return 2 - beta * mp.log((beta + 1) / (beta - 1))


def cf2_paper_eq18(x):
    x = mp.mpc(x)
    w = mp.sqrt(1 - x * x)
    acos = -1j * mp.log(x + 1j * w)
    return 1 - mp.pi / (2 * x) + w * acos / x


def cf3_feynman(x, a, b):
    x, a, b = mp.mpc(x), mp.mpc(a), mp.mpc(b)
    f = lambda al: mp.log(1 + al * (1 - al) * x / (al * a + (1 - al) * b))
    return -mp.quad(f, [0, 0.25, 0.5, 0.75, 1])


def rational_poles(M2, a, b):
    """(u + M2)/(u^2 + a u + b) = sum_r R_r / (u - u_r)."""
    disc = mp.sqrt(mp.mpc(a * a - 4 * b))
    u1, u2 = (-a + disc) / 2, (-a - disc) / 2
    R1, R2 = (u1 + M2) / (u1 - u2), (u2 + M2) / (u2 - u1)
    return [(u1, R1), (u2, R2)]


def cf3_rational(x, m1sq, M2, a, b):
    return sum(R * cf3_feynman(x, m1sq, -u) for (u, R) in rational_poles(M2, a, b))


def in_parabola_R2(x, m2=1.0, shrink=0.0):
    """REAL contour equals the continuation iff Re x > (Im x)^2/(4 m^2) - m^2 (R2,
    derived from eq. (23); 'parabola-shaped region on the right')."""
    x = complex(x)
    return x.real - shrink > x.imag ** 2 / (4 * m2) - m2


def angular_B_massive(x, y, mu):
    """Paper eq. (22), term B, in the continuum for a massive line 2 with mass^2 mu:
       B = (y + mu) [ pi (A - r) / b^2 - (pi/2)/(y + mu) ],  A = x + y + mu, b = 2 sqrt(x) sqrt(y), r^2 = A^2 - b^2,
    from the textbook integral  int_-1^1 sqrt(1-z^2)/(A - b z) dz = pi (A - r)/b^2  with the root r for which
    |A - r| < |A + r| (the branch that decays like pi/(2A); it is analytic in A/b off [-1, 1], i.e. off the cut of
    eq. (25))."""
    x, y, mu = mp.mpc(x), mp.mpc(y), mp.mpc(mu)
    A, b = x + y + mu, 2 * mp.sqrt(x) * mp.sqrt(y)
    r = mp.sqrt(A * A - b * b)
    if (mp.conj(A) * r).real < 0:
        r = -r
    return (y + mu) * (mp.pi * (A - r) / b ** 2 - mp.pi / 2 / (y + mu))


def bubble_d3(x, m=1.0):
    """Equal-mass bubble in d = 3, subtracted at x = 0, normalised int d^3k/(2 pi)^3:
         G(x) = arctan(sqrt(x)/(2m)) / (4 pi sqrt(x)) - 1/(8 pi m)
    (textbook; arctan w = ln((1 + i w)/(1 - i w))/(2i); even in sqrt(x); cut x <= -4 m^2 like CF1).  In the
    variables of the scan: c0 = 1/(8 pi^2), radial measure dy y^(1/2), angular measure dz (d^3k = 1/2 y^(1/2) dy 2 pi dz)."""
    x, m = mp.mpc(x), mp.mpf(m)
    if x == 0:
        return mp.mpc(0)
    w = mp.sqrt(x) / (2 * m)
    at = mp.log((1 + 1j * w) / (1 - 1j * w)) / 2j
    return at / (4 * mp.pi * mp.sqrt(x)) - 1 / (8 * mp.pi * m)
