"""Closed forms that pin the oracle (GR textbook facts and the paper's own formulas).

Nothing here is an implementation of the method: these are the independent facts the oracle is
checked against.  G = c = M = 1.
Citations: PAPER.md = /root/reference/PAPER.md (arXiv:1706.07062).
"""
from __future__ import annotations

import numpy as np


# ---- F1, F2: horizon, ergosphere, circular photon orbits (eq. 19-21) ----------

def r_plus(a):
    return 1.0 + np.sqrt(1.0 - a * a)


def r_minus(a):
    return 1.0 - np.sqrt(1.0 - a * a)


def r_ergo(a, theta):
    return 1.0 + np.sqrt(1.0 - a * a * np.cos(theta) ** 2)


def r_photon_prograde(a):
    return 2.0 * (1.0 + np.cos(2.0 / 3.0 * np.arccos(-abs(a))))


def r_photon_retrograde(a):
    return 2.0 * (1.0 + np.cos(2.0 / 3.0 * np.arccos(abs(a))))


# ---- F3, F4: spherical photon orbits (Teo 2003 / Bardeen 1973), E = 1 ----------------------------

def teo_phi_q(a, r):
    """Normalised L_z (Phi) and Carter constant (Q) of the spherical photon orbit of radius r."""
    phi = -(r ** 3 - 3.0 * r ** 2 + a * a * r + a * a) / (a * (r - 1.0))
    q = -(r ** 3) * (r ** 3 - 6.0 * r ** 2 + 9.0 * r - 4.0 * a * a) / (a * a * (r - 1.0) ** 2)
    return phi, q


def max_abs_costheta(a, phi, q):
    """sqrt(u0), u0 the positive root of a^2 u^2 + (Q + Phi^2 - a^2) u - Q = 0  (Theta(theta) = 0)."""
    b = q + phi * phi - a * a
    u0 = (-b + np.sqrt(b * b + 4.0 * a * a * q)) / (2.0 * a * a)
    return np.sqrt(u0)


def equatorial_first_integrals(a, r, E, Lz, Q, mu2=0.0):
    """BL (= spherical KS when u^r = 0) u^t, u^phi, u^theta at theta = pi/2, 'moving upward'.

    Standard first integrals of Kerr geodesics at theta = pi/2 (rho^2 = r^2):
      T = E (r^2+a^2) - a Lz ;  u^t = [-a(aE - Lz) + (r^2+a^2) T/Delta]/r^2 ;
      u^phi = [-(aE - Lz) + a T/Delta]/r^2 ;  u^theta = -sqrt(Q)/r^2.
    """
    delta = r * r - 2.0 * r + a * a
    T = E * (r * r + a * a) - a * Lz
    ut = (-a * (a * E - Lz) + (r * r + a * a) * T / delta) / (r * r)
    uphi = (-(a * E - Lz) + a * T / delta) / (r * r)
    uth = -np.sqrt(max(Q, 0.0)) / (r * r)
    return ut, uphi, uth


def ks_state_on_equator(a, r, ut, uphi, uth, phi_ks=0.0, ur=0.0):
    """Cartesian KS 8-vector of a particle at (r, theta=pi/2, phi_KS) with u^r = 0.

    x + i y = (r + i a) e^{i phi};  with u^r = 0 the BL and KS components of u^t, u^phi coincide
    (F11: the two coordinate systems differ by functions of r only)."""
    assert ur == 0.0
    x = r * np.cos(phi_ks) - a * np.sin(phi_ks)
    y = r * np.sin(phi_ks) + a * np.cos(phi_ks)
    return np.array([0.0, x, y, 0.0, ut, -y * uphi, x * uphi, -r * uth])


def spherical_photon_state(a, r):
    """Initial data of the paper's Table 1 tests: E = 1, equator, moving upward."""
    phi, q = teo_phi_q(a, r)
    ut, uphi, uth = equatorial_first_integrals(a, r, 1.0, phi, q)
    return ks_state_on_equator(a, r, ut, uphi, uth), phi, q


# ---- F6, F7: Bardeen shadow boundary and Carter's radial potential -------------------------------

def bardeen_curve(a, inc, n=200001):
    """Shadow boundary for an observer at infinity at inclination inc (upper half, beta >= 0).

    alpha = -xi / sin i ; beta = sqrt(eta + a^2 cos^2 i - xi^2 cot^2 i), (xi, eta) = teo_phi_q(a, r),
    r in [r_p, r_r] where beta^2 >= 0.  a = 0: circle of radius sqrt(27)."""
    if a == 0.0:
        t = np.linspace(0.0, np.pi, n)
        return np.sqrt(27.0) * np.cos(t), np.sqrt(27.0) * np.sin(t)
    r = np.linspace(r_photon_prograde(a), r_photon_retrograde(a), n)
    xi, eta = teo_phi_q(a, r)
    b2 = eta + a * a * np.cos(inc) ** 2 - xi * xi / np.tan(inc) ** 2
    ok = b2 >= 0.0
    return -xi[ok] / np.sin(inc), np.sqrt(b2[ok])


def bardeen_edges_on_axis(a, inc):
    """The two alpha values where the shadow boundary crosses beta = 0 (bisection on beta^2(r))."""
    def b2(r):
        xi, eta = teo_phi_q(a, r)
        return eta + a * a * np.cos(inc) ** 2 - xi * xi / np.tan(inc) ** 2

    def root(lo, hi):
        flo = b2(lo)
        for _ in range(200):
            mid = 0.5 * (lo + hi)
            if (b2(mid) > 0) == (flo > 0):
                lo = mid
            else:
                hi = mid
        return 0.5 * (lo + hi)

    rp, rr = r_photon_prograde(a), r_photon_retrograde(a)
    rs = np.linspace(rp, rr, 20001)
    rmax = rs[np.argmax(b2(rs))]
    r1 = root(rp - 1e-9 if b2(rp) > 0 else rp, rmax) if b2(rp) <= 0 else rp
    r2 = root(rr, rmax) if b2(rr) <= 0 else rr
    return sorted([-teo_phi_q(a, r1)[0] / np.sin(inc), -teo_phi_q(a, r2)[0] / np.sin(inc)])


def carter_R_coeffs(a, xi, eta):
    """R(r) = (r^2+a^2-a xi)^2 - Delta [eta + (xi-a)^2] as a quartic (null, E = 1), highest power first."""
    K = eta + (xi - a) ** 2
    return [1.0, 0.0, a * a - xi * xi - eta, 2.0 * K, -a * a * eta]


def captured_by_potential(a, xi, eta, r_start):
    """True iff an inward-moving photon with conserved (xi, eta) has no radial turning point in
    (r_plus, r_start): R(r) > 0 throughout.  Independent of any ODE solve."""
    roots = np.roots(carter_R_coeffs(a, xi, eta))
    rp = r_plus(a)
    for z in roots:
        if abs(z.imag) < 1e-9 * max(1.0, abs(z.real)) and rp < z.real < r_start:
            return False
    return True


def distance_to_bardeen(a, inc, alpha, beta, curve=None):
    """Distance in the (alpha, beta) plane from points to the critical curve (both halves)."""
    ca, cb = curve if curve is not None else bardeen_curve(a, inc)
    alpha = np.atleast_1d(alpha)
    beta = np.abs(np.atleast_1d(beta))
    out = np.empty(alpha.shape)
    for i in range(alpha.size):
        out.flat[i] = np.sqrt(np.min((ca - alpha.flat[i]) ** 2 + (cb - beta.flat[i]) ** 2))
    return out


# ---- F8-F10: circular equatorial time-like orbits (Bardeen, Press & Teukolsky 1972) --------------

def circular_orbit(a, r, s=+1):
    """Omega, E, Lz, u^t of the circular equatorial orbit (s=+1 prograde, -1 retrograde)."""
    omega = s / (r ** 1.5 + s * a)
    D = r ** 0.75 * np.sqrt(r ** 1.5 - 3.0 * r ** 0.5 + 2.0 * s * a)
    E = (r ** 1.5 - 2.0 * r ** 0.5 + s * a) / D
    Lz = s * (r * r - 2.0 * s * a * r ** 0.5 + a * a) / D
    ut = (1.0 - 2.0 / r + 4.0 * a * omega / r - (r * r + a * a + 2.0 * a * a / r) * omega ** 2) ** -0.5
    return omega, E, Lz, ut


def circular_orbit_state(a, r, s=+1, vz=0.0):
    omega, E, Lz, ut = circular_orbit(a, r, s)
    st = ks_state_on_equator(a, r, ut, omega * ut, 0.0)
    st[7] = vz
    return st


def r_isco(a, s=+1):
    z1 = 1.0 + (1.0 - a * a) ** (1.0 / 3.0) * ((1.0 + a) ** (1.0 / 3.0) + (1.0 - a) ** (1.0 / 3.0))
    z2 = np.sqrt(3.0 * a * a + z1 * z1)
    return 3.0 + z2 - s * np.sqrt((3.0 - z1) * (3.0 + z1 + 2.0 * z2))


def vertical_epicyclic(a, r, s=+1):
    omega = s / (r ** 1.5 + s * a)
    return abs(omega) * np.sqrt(1.0 - 4.0 * s * a * r ** -1.5 + 3.0 * a * a / (r * r))


# ---- F11: Kerr-Schild <-> Boyer-Lindquist (replaces the paper's missing Appendix) --

def bl_to_ks(a, X, u):
    """Map a BL point X = (t, r, theta, phi_BL) and contravariant u to Cartesian KS (8-vector).

    dt_KS = dt_BL + (2 r / Delta) dr ; dphi_KS = dphi_BL + (a / Delta) dr ;
    x + i y = (r + i a) sin(theta) e^{i phi_KS} ; z = r cos(theta)."""
    t, r, th, ph = X
    rp, rm = r_plus(a), r_minus(a)
    delta = r * r - 2.0 * r + a * a
    if rp != rm:
        t_ks = t + 2.0 / (rp - rm) * (rp * np.log(abs(r - rp)) - rm * np.log(abs(r - rm)))
        ph_ks = ph + a / (rp - rm) * np.log(abs((r - rp) / (r - rm)))
    else:
        raise ValueError("extremal case not needed")
    sth, cth = np.sin(th), np.cos(th)
    cp, sp = np.cos(ph_ks), np.sin(ph_ks)
    x = (r * cp - a * sp) * sth
    y = (r * sp + a * cp) * sth
    z = r * cth
    # Jacobian d(t_ks, x, y, z) / d(t, r, theta, phi_BL)
    J = np.zeros((4, 4))
    J[0, 0] = 1.0
    J[0, 1] = 2.0 * r / delta
    dph_dr = a / delta
    J[1, 1] = cp * sth + (-y) * dph_dr
    J[2, 1] = sp * sth + (x) * dph_dr
    J[3, 1] = cth
    J[1, 2] = (r * cp - a * sp) * cth
    J[2, 2] = (r * sp + a * cp) * cth
    J[3, 2] = -r * sth
    J[1, 3] = -y
    J[2, 3] = x
    uk = J @ np.asarray(u, dtype=float)
    return np.array([t_ks, x, y, z, *uk]), J


def ks_to_bl_position(a, pos):
    """(r, theta, phi_BL) of a Cartesian KS point (x, y, z)."""
    x, y, z = pos
    R2 = x * x + y * y + z * z
    w = R2 - a * a
    r = np.sqrt(0.5 * (w + np.sqrt(w * w + 4.0 * a * a * z * z)))
    th = np.arccos(np.clip(z / r, -1.0, 1.0))
    ph_ks = np.arctan2(y, x) - np.arctan2(a, r)
    rp, rm = r_plus(a), r_minus(a)
    ph_bl = ph_ks - a / (rp - rm) * np.log(abs((r - rp) / (r - rm))) if rp != rm else ph_ks
    return r, th, ph_bl
