"""Helpers shared by the image-plane tests (oracle pins and GPU parity): the critical-curve band of
DESIGN R11 and the ODE-free capture classifier built on Carter's radial potential (closed_forms F6/F7).

The conserved (xi, eta) = (Lz/E, Q/E^2) of each ray are taken from the ORACLE's invariants of the
initial state; everything after that is closed form."""
import numpy as np

import closed_forms as cf
import oracle


def ray_constants(state):
    """(xi_run, eta) of every ray of an oracle State (run spacetime, spin state.a_eff)."""
    E, Lz, Q, norm = oracle.invariants(state)
    return Lz / E, Q / (E * E), E, norm


def asymptotic_image_point(a_run, inc, xi_run, eta, beta_sign):
    """Bardeen's image-plane point of a ray with conserved (xi, eta) for an observer at infinity.
    In the run spacetime (spin a_run = -a, DESIGN R3) the physical xi is -xi_run, so alpha = xi_run/sin i."""
    alpha = xi_run / np.sin(inc)
    b2 = eta + a_run * a_run * np.cos(inc) ** 2 - xi_run * xi_run / np.tan(inc) ** 2
    return alpha, np.sign(beta_sign) * np.sqrt(np.maximum(b2, 0.0))


def band_distance(a_phys, inc, alpha_inf, beta_inf):
    """Distance of every ray to the critical curve in the asymptotic image plane (vectorised, chunked)."""
    ca, cb = cf.bardeen_curve(abs(a_phys), inc, n=100001)
    if a_phys < 0:
        ca = -ca
    al = np.asarray(alpha_inf).ravel()
    be = np.abs(np.asarray(beta_inf).ravel())
    out = np.empty(al.size)
    # coarse pre-selection keeps this O(n * few) instead of O(n * 1e5)
    step = 64
    cca, ccb = ca[::step], cb[::step]
    for lo in range(0, al.size, 4096):
        hi = min(lo + 4096, al.size)
        d2 = (cca[None, :] - al[lo:hi, None]) ** 2 + (ccb[None, :] - be[lo:hi, None]) ** 2
        j = np.argmin(d2, axis=1) * step
        best = np.full(hi - lo, np.inf)
        for off in range(-step, step + 1):
            jj = np.clip(j + off, 0, ca.size - 1)
            best = np.minimum(best, (ca[jj] - al[lo:hi]) ** 2 + (cb[jj] - be[lo:hi]) ** 2)
        out[lo:hi] = np.sqrt(best)
    return out.reshape(np.shape(alpha_inf))


def potential_mask(a_run, xi_run, eta, r_start):
    """True where Carter's radial potential has no turning point between r_plus and r_start (captured)."""
    xi_run = np.asarray(xi_run).ravel()
    eta = np.asarray(eta).ravel()
    out = np.empty(xi_run.size, dtype=bool)
    for k in range(xi_run.size):
        out[k] = cf.captured_by_potential(a_run, xi_run[k], eta[k], r_start)
    return out


def pixel_grid(cfg):
    """(alpha, beta) of every pixel in index order k*nx + j (DESIGN R1: pixel centres)."""
    al = -cfg.fov + (np.arange(cfg.nx) + 0.5) * (2.0 * cfg.fov / cfg.nx)
    be = -cfg.fov + (np.arange(cfg.ny) + 0.5) * (2.0 * cfg.fov / cfg.ny)
    A, B = np.meshgrid(al, be)
    return A.ravel(), B.ravel()


def classify_image(cfg, state0):
    """For the initial oracle state of an image: band distance d (DESIGN R11) and the F7 capture mask."""
    xi, eta, E, norm = ray_constants(state0)
    _, beta = pixel_grid(cfg)
    a_inf, b_inf = asymptotic_image_point(state0.a_eff, cfg.inclination, xi, eta, np.where(beta >= 0, 1.0, -1.0))
    if cfg.a == 0.0:
        d = np.abs(np.sqrt(xi * xi + eta) - np.sqrt(27.0))
    else:
        d = band_distance(cfg.a, cfg.inclination, a_inf, b_inf)
    r0 = np.array([oracle.ks_r(state0.a_eff, *state0.q[1:4, k]) for k in range(0, state0.n, max(1, state0.n // 64))])
    mask = potential_mask(state0.a_eff, xi, eta, r0.min())
    return d, mask


def axis_approach(state0):
    """sin(theta_min): how close each null ray's polar motion comes to the spin axis, from its conserved
    (xi, eta) alone.  Theta(theta) = eta + cos^2 (a^2 - xi^2 / sin^2) vanishes at the polar turning points
    (Carter 1968; E = 1):  a^2 u^2 + (eta + xi^2 - a^2) u - eta = 0 for u = cos^2 at the turning point
    nearest the axis (the larger root; for the few vortical rays, eta < 0, eta is clamped to 0 in the
    discriminant, which only moves them further from the threshold the tests use)."""
    xi, eta, E, norm = ray_constants(state0)
    a = state0.a_eff
    if a == 0.0:
        u0 = np.clip(eta / np.maximum(eta + xi * xi, 1e-300), 0.0, 1.0)   # cos^2 = eta / (eta + xi^2)
    else:
        b = eta + xi * xi - a * a
        u0 = (-b + np.sqrt(b * b + 4.0 * a * a * np.maximum(eta, 0.0))) / (2.0 * a * a)
    return np.sqrt(np.clip(1.0 - u0, 0.0, 1.0))
