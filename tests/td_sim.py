"""Time-domain simulation of TDI X used to pin the oracle's frequency-domain response (pin P9).

Independent of the oracle's response code: it works in the time domain with exact Keplerian
spacecraft orbits (Kepler's equation solved numerically), the textbook one-way Doppler response

    y_sr(t) = n.[H(t - L/c - k.p_s/c) - H(t - k.p_r/c)].n / (2 (1 - k.n)),   H = h_+ e_+ + h_x e_x,

(the time-domain statement behind PAPER.md:196 Eq. 15: antenna factor F(t) times a delayed h), and
first-generation Michelson X built with explicit delays L/c, 2L/c, 3L/c ("a sum of
time-delayed single-arm responses").  The only thing taken from the oracle is the scalar phase
function Psi_0(f) and t_f, from which the time-domain chirp is obtained by the stationary-phase
Legendre transform  Phi(t_f) = 2 pi f t_f - Psi_0(f) - pi/4,  a(t_f) = 2 f^(-7/6) sqrt(df/dt).
"""
import numpy as np
from scipy.interpolate import CubicHermiteSpline, CubicSpline

AU = 149597870700.0
YR = 31557600.0
C = 299792458.0


def kepler_positions(t, L, kappa=0.0, lam=0.0):
    """Exact Keplerian LISA orbits: ellipses with a = 1 AU, eccentricity e = L/(2 sqrt(3) AU),
    inclination sqrt(3) e, phased 120 degrees apart.  Returns [3][3][len(t)] (spacecraft, xyz, time)."""
    t = np.atleast_1d(np.asarray(t, dtype=np.float64))
    e = L / (2.0 * np.sqrt(3.0) * AU)
    out = np.empty((3, 3, t.shape[0]))
    al = 2.0 * np.pi * t / YR + kappa
    for n in range(3):
        be = 2.0 * np.pi * n / 3.0 + lam
        m = al - be
        psi = m.copy()
        for _ in range(6):                        # Newton on psi - e sin psi = m
            psi = psi - (psi - e * np.sin(psi) - m) / (1.0 - e * np.cos(psi))
        gam = 2.0 * np.arctan2(np.sqrt(1.0 + e) * np.sin(0.5 * psi), np.sqrt(1.0 - e) * np.cos(0.5 * psi))
        r = AU * (1.0 - e * e) / (1.0 + e * np.cos(gam))
        inc = np.sqrt(3.0) * e
        out[n, 0] = r * (np.cos(inc) * np.cos(be) * np.cos(gam) - np.sin(be) * np.sin(gam))
        out[n, 1] = r * (np.cos(inc) * np.sin(be) * np.cos(gam) + np.cos(be) * np.sin(gam))
        out[n, 2] = -r * np.sin(inc) * np.cos(gam)
    return out


class Chirp:
    """h_P(t) = |c_P| a(t) cos(Phi(t) + arg c_P) whose SPA Fourier transform is c_P f^(-7/6) exp(-i Psi_0(f))."""

    def __init__(self, f_nodes, psi_nodes, tf_nodes):
        f, psi, tf = map(np.asarray, (f_nodes, psi_nodes, tf_nodes))
        assert np.all(np.diff(tf) > 0)
        phi = 2.0 * np.pi * f * tf - psi - np.pi / 4.0
        self.t0, self.t1 = tf[0], tf[-1]
        self._phi = CubicHermiteSpline(tf, phi, 2.0 * np.pi * f)      # dPhi/dt = 2 pi f exactly
        self._f = CubicSpline(tf, f)
        fdot = 1.0 / np.gradient(tf, f, edge_order=2)
        self._amp = CubicSpline(tf, 2.0 * f ** (-7.0 / 6.0) * np.sqrt(fdot))

    def h(self, t, c_plus, c_cross):
        ph, a = self._phi(t), self._amp(t)
        return (abs(c_plus) * a * np.cos(ph + np.angle(c_plus)),
                abs(c_cross) * a * np.cos(ph + np.angle(c_cross)))


def tdi_michelson_time_domain(t, chirp, c_plus, c_cross, theta, phi, L, vertex=0):
    """First-generation Michelson combination centred on spacecraft `vertex` (0, 1, 2 <-> X, Y, Z) from its four
    one-way links with explicit delays; Y and Z are X with the spacecraft relabelled cyclically."""
    st, ct, sp, cp = np.sin(theta), np.cos(theta), np.sin(phi), np.cos(phi)
    k = np.array([-st * cp, -st * sp, -ct])
    u = np.array([ct * cp, ct * sp, -st])
    v = np.array([sp, -cp, 0.0])
    Lc = L / C

    def link(s, r, tt):
        p = kepler_positions(tt, L)
        ps, pr = p[s], p[r]
        n = (pr - ps) / L
        kn = k @ n
        un, vn = u @ n, v @ n
        xi_p, xi_c = un * un - vn * vn, 2.0 * un * vn
        hp_s, hc_s = chirp.h(tt - Lc - (k @ ps) / C, c_plus, c_cross)
        hp_r, hc_r = chirp.h(tt - (k @ pr) / C, c_plus, c_cross)
        return (xi_p * (hp_s - hp_r) + xi_c * (hc_s - hc_r)) / (2.0 * (1.0 - kn))

    # spacecraft indices 0,1,2 <-> 1,2,3;  y_sr: photon leaves s, arrives at r.  For X: a = 0, b = 1, c = 2
    a, b, c = vertex, (vertex + 1) % 3, (vertex + 2) % 3
    x = (link(c, a, t) + link(a, c, t - Lc) + link(b, a, t - 2 * Lc) + link(a, b, t - 3 * Lc)
         - link(b, a, t) - link(a, b, t - Lc) - link(c, a, t - 2 * Lc) - link(a, c, t - 3 * Lc))
    return x


def tdi_x_time_domain(t, chirp, c_plus, c_cross, theta, phi, L):
    """X(t) from the four one-way links with explicit delays."""
    return tdi_michelson_time_domain(t, chirp, c_plus, c_cross, theta, phi, L, 0)


class PhysicalBinary:
    """Time-domain strain of a quasi-circular binary from the quadrupole formula, with NOTHING of App. A-B in it (pin P20):
    two point masses on a circular orbit of phase Phi(t)/2 about the unit vector Lhat, seen at distance D,

        h_ij(t) = -A(t) [ (e1 e1 - e2 e2)_ij cos Phi(t) + (e1 e2 + e2 e1)_ij sin Phi(t) ],
        A(t) = 4 (G M_c / c^3)^(5/3) (pi f(t))^(2/3) / (D / c),

    (x(t) = e1 cos(Phi/2) + e2 sin(Phi/2) the separation direction, e1, e2 orthonormal in the orbital plane, e1 x e2 = Lhat;
    h_ij = (2 G / c^4 D) d^2 Q_ij / dt^2 at leading order, M_c^(5/3) = mu M^(2/3), omega = pi f), projected on the sky basis
    of the propagation direction k: h_+ = (u.h.u - v.h.v)/2, h_x = u.h.v.  The orientation is given physically: iota = angle
    between Lhat and k (k points from the source to the observer), pol = angle of Lhat's sky projection from u towards v.
    Several (D, iota, pol, phi0) sets are carried at once: h() returns arrays [n_sets][len(t)], so that the links of
    tdi_michelson_time_domain (whose cost is the Keplerian orbits) are evaluated once."""

    def __init__(self, chirp, chirp_mass_s, k, u, v, sets):
        self.chirp, self.tau = chirp, float(chirp_mass_s)
        self.coef = []
        for (dist_s, iota, pol, phi0) in sets:
            lhat = np.cos(iota) * k + np.sin(iota) * (np.cos(pol) * u + np.sin(pol) * v)
            e1 = np.cross(lhat, k)
            e1 = e1 / np.linalg.norm(e1)
            e2 = np.cross(lhat, e1)

            def comp(a, b, e1=e1, e2=e2):               # (cos, sin) coefficients of a.h.b / (-A)
                return ((a @ e1) * (b @ e1) - (a @ e2) * (b @ e2), (a @ e1) * (b @ e2) + (a @ e2) * (b @ e1))
            uu, vv, uv = comp(u, u), comp(v, v), comp(u, v)
            self.coef.append((dist_s, phi0, 0.5 * (uu[0] - vv[0]), 0.5 * (uu[1] - vv[1]), uv[0], uv[1]))

    def h(self, t, c_plus=None, c_cross=None):
        phi, f = self.chirp._phi(t), self.chirp._f(t)
        amp = 4.0 * self.tau ** (5.0 / 3.0) * (np.pi * f) ** (2.0 / 3.0)
        hp, hc = [], []
        for (dist_s, phi0, pc, ps, cc, cs) in self.coef:
            co, si = np.cos(phi + phi0), np.sin(phi + phi0)
            hp.append(-(amp / dist_s) * (pc * co + ps * si))
            hc.append(-(amp / dist_s) * (cc * co + cs * si))
        return np.array(hp), np.array(hc)
