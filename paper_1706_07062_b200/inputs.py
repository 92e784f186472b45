"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the oracle tests and the CUDA path (tests, bench.py).  It holds none of the
method's arithmetic: no Kerr-Schild metric, no geodesic right-hand side, no Runge-Kutta, no
invariants.  What it does hold is (i) the scalar parameters of each config, (ii) a counter-based
random generator (splitmix64), and (iii) the textbook Kerr orbital mechanics (Boyer-Lindquist first
integrals, Carter's radial potential) needed to turn orbital elements (p, e, cos iota) into explicit
Cartesian 8-vectors.  The 8-vectors are produced once, in double, and the same array is handed to
the oracle and to ``gray2_init_timelike``, so the generator is not part of the parity surface.

The paper measures on its own synthetic image of rays; no public data set is
involved, and none is stood in for.  Recipes: DESIGN.md "Input recipe".
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

_M64 = (1 << 64) - 1


def splitmix64_uniform(seed: int, counters: np.ndarray) -> np.ndarray:
    """u in [0,1) from the splitmix64 finaliser of (seed + (counter+1) * golden), vectorised."""
    c = np.asarray(counters, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = np.uint64(seed & _M64) + (c + np.uint64(1)) * np.uint64(0x9E3779B97F4A7C15)
        z ^= z >> np.uint64(30)
        z *= np.uint64(0xBF58476D1CE4E5B9)
        z ^= z >> np.uint64(27)
        z *= np.uint64(0x94D049BB133111EB)
        z ^= z >> np.uint64(31)
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


# ---------------------------------------------------------------------------------------------------
# Config table (BASELINE.json "configs", restated as concrete scalars)
# ---------------------------------------------------------------------------------------------------

@dataclass(frozen=True)
class NullImageConfig:
    name: str
    a: float
    r_obs: float
    inclination_deg: float
    fov: float            # half-width in alpha and beta [M]
    nx: int
    ny: int
    eta: float = 0.01
    r_escape: float = 1100.0
    max_steps: int = 20000
    capture_factor: float = 1.01

    @property
    def inclination(self) -> float:
        return math.radians(self.inclination_deg)

    @property
    def n(self) -> int:
        return self.nx * self.ny

    def scaled(self, nx: int, ny: int | None = None) -> "NullImageConfig":
        """Same field of view sampled on a coarser (or finer) pixel grid."""
        return NullImageConfig(self.name + "@%d" % nx, self.a, self.r_obs, self.inclination_deg, self.fov,
                               nx, nx if ny is None else ny, self.eta, self.r_escape, self.max_steps,
                               self.capture_factor)


CFG1_NULL = NullImageConfig("cfg1a-schwarzschild-64", 0.0, 100.0, 60.0, 10.0, 64, 64, r_escape=150.0)
CFG2_NULL = NullImageConfig("cfg2-kerr0.99-512", 0.99, 1000.0, 17.0, 12.0, 512, 512)
CFG3_NULL = NullImageConfig("cfg3-kerr0.9375-1024", 0.9375, 1000.0, 60.0, 15.0, 1024, 1024)
CFG5_NULL = NullImageConfig("cfg5-kerr0.5-4096", 0.5, 1000.0, 30.0, 20.0, 4096, 4096)

CFG1_ORBITS = dict(name="cfg1b-schwarzschild-orbits", a=0.0, n=16, seed=1706, h_fixed=0.5, max_steps=5000)
CFG4_ENSEMBLE = dict(name="cfg4-kerr0.7-ensemble", a=0.7, n=1 << 20, seed=7062, h_fixed=0.5,
                     max_steps=100000, p_range=(8.0, 50.0), e_range=(0.0, 0.8))


# ---------------------------------------------------------------------------------------------------
# cfg1b: 16 seeded circular time-like orbits in Schwarzschild, tilted planes
# ---------------------------------------------------------------------------------------------------

def cfg1_orbits(n: int = 16, seed: int = 1706):
    """Circular geodesic orbits at r0 in (6, 20], a = 0, random orbital plane and phase.

    Schwarzschild circular orbit: Omega = r0^-3/2, u^t = (1 - 3/r0)^-1/2 (textbook).  In the a = 0
    Kerr-Schild (ingoing Eddington-Finkelstein) Cartesian chart a circular orbit has u^r = 0, so its
    components equal the Schwarzschild ones.  Returns (xu8[n,8], r0[n])."""
    k = np.arange(n, dtype=np.uint64)
    u = [splitmix64_uniform(seed, k * np.uint64(4) + np.uint64(j)) for j in range(4)]
    r0 = 20.0 - 14.0 * u[0]                       # (6, 20]
    cosi = -1.0 + 2.0 * u[1]
    node = 2.0 * math.pi * u[2]
    phase = 2.0 * math.pi * u[3]
    sini = np.sqrt(1.0 - cosi * cosi)
    # orthonormal basis of the orbital plane: e1 along the line of nodes, e2 = n x e1
    e1 = np.stack([np.cos(node), np.sin(node), np.zeros(n)], axis=1)
    nrm = np.stack([sini * np.sin(node), -sini * np.cos(node), cosi], axis=1)
    e2 = np.cross(nrm, e1)
    ut = 1.0 / np.sqrt(1.0 - 3.0 / r0)
    omega = r0 ** -1.5
    pos = r0[:, None] * (np.cos(phase)[:, None] * e1 + np.sin(phase)[:, None] * e2)
    vel = (r0 * omega * ut)[:, None] * (-np.sin(phase)[:, None] * e1 + np.cos(phase)[:, None] * e2)
    xu8 = np.zeros((n, 8))
    xu8[:, 1:4] = pos
    xu8[:, 4] = ut
    xu8[:, 5:8] = vel
    return xu8, r0


# ---------------------------------------------------------------------------------------------------
# cfg4: bound Kerr orbits from (p, e, cos iota)
# ---------------------------------------------------------------------------------------------------

def _R_poly(a, E, L, c):
    """Coefficients (r^4..r^0) of Carter's radial potential for mu = 1 with Lz = L c, Q = L^2 (1-c^2):
    R(r) = [E(r^2+a^2) - a Lz]^2 - Delta [r^2 + (Lz - aE)^2 + Q]."""
    Lz = L * c
    Q = L * L * (1.0 - c * c)
    c4 = E * E - 1.0
    c3 = 2.0 * np.ones_like(E)
    c2 = a * a * (E * E - 1.0) - Lz * Lz - Q
    c1 = 2.0 * ((a * E - Lz) ** 2 + Q)
    c0 = -a * a * Q
    return c4, c3, c2, c1, c0


def _polyval(cs, r):
    out = np.zeros_like(r)
    for ck in cs:
        out = out * r + ck
    return out


def _divided_difference(cs, r1, r2):
    """[R(r2) - R(r1)] / (r2 - r1) for a quartic, exact also when r1 == r2 (-> R'(r1))."""
    c4, c3, c2, c1, _ = cs
    s1 = np.ones_like(r1)
    s2 = r1 + r2
    s3 = r1 * r1 + r1 * r2 + r2 * r2
    s4 = (r1 + r2) * (r1 * r1 + r2 * r2)
    return c4 * s4 + c3 * s3 + c2 * s2 + c1 * s1


def solve_orbit_constants(a, p, e, cosi, iters=60):
    """(E, Lz, Q) of the bound orbit with turning points r_p = p/(1+e), r_a = p/(1-e) and
    cos iota = Lz / sqrt(Lz^2 + Q).  Newton in (E, L) on R(r_p) = 0 and the divided difference
    [R(r_a)-R(r_p)]/(r_a-r_p) = 0, started from the Schwarzschild closed form.  Returns E, Lz, Q, ok."""
    p, e, cosi = (np.asarray(v, dtype=np.float64) for v in (p, e, cosi))
    rp, ra = p / (1.0 + e), p / (1.0 - e)
    den = p - 3.0 - e * e
    E = np.sqrt(np.maximum(((p - 2.0) ** 2 - 4.0 * e * e) / (p * den), 1e-6))
    L = np.sqrt(np.maximum(p * p / den, 1e-6))

    def F(E, L):
        cs = _R_poly(a, E, L, cosi)
        return _polyval(cs, rp), _divided_difference(cs, rp, ra)

    ok = np.ones(p.shape, dtype=bool)
    for _ in range(iters):
        f1, f2 = F(E, L)
        dE, dL = 1e-7, 1e-7 * np.maximum(L, 1.0)
        f1e, f2e = F(E + dE, L)
        f1l, f2l = F(E, L + dL)
        j11, j21 = (f1e - f1) / dE, (f2e - f2) / dE
        j12, j22 = (f1l - f1) / dL, (f2l - f2) / dL
        det = j11 * j22 - j12 * j21
        with np.errstate(all="ignore"):
            sE = (f1 * j22 - f2 * j12) / det
            sL = (j11 * f2 - j21 * f1) / det
        bad = ~np.isfinite(sE) | ~np.isfinite(sL)
        sE = np.where(bad, 0.0, sE)
        sL = np.where(bad, 0.0, sL)
        ok &= ~bad
        # damp large Newton steps
        sE = np.clip(sE, -0.05, 0.05)
        sL = np.clip(sL, -1.0, 1.0)
        E, L = E - sE, L - sL
        if _ >= 4 and float(np.max(np.abs(sE))) < 1e-15 and float(np.max(np.abs(sL) / np.maximum(L, 1.0))) < 1e-15:
            break
    f1, f2 = F(E, L)
    scale = rp ** 4
    ok &= (np.abs(f1) < 1e-9 * scale) & (np.abs(f2) < 1e-9 * scale / rp) & (L > 0) & np.isfinite(E)
    Lz = L * cosi
    Q = L * L * (1.0 - cosi * cosi)
    return E, Lz, Q, ok


def orbit_is_bound(a, E, Lz, Q, rp, ra, nsamp=64):
    """E < 1, R'(r_p) > 0, R'(r_a) < 0 and R > 0 on nsamp radii inside (r_p, r_a)."""
    c4 = E * E - 1.0
    c3 = 2.0 * np.ones_like(E)
    c2 = a * a * (E * E - 1.0) - Lz * Lz - Q
    c1 = 2.0 * ((a * E - Lz) ** 2 + Q)
    c0 = -a * a * Q
    cs = (c4, c3, c2, c1, c0)
    dcs = (4.0 * c4, 3.0 * c3, 2.0 * c2, c1)
    ok = (E < 1.0) & (_polyval(dcs, rp) > 0.0)
    wide = ra > rp * (1.0 + 1e-9)
    ok &= np.where(wide, _polyval(dcs, ra) < 0.0, True)
    for k in range(1, nsamp + 1):
        r = rp + (ra - rp) * (k / (nsamp + 1.0))
        ok &= np.where(wide, _polyval(cs, r) > 0.0, True)
    # circular limit (e -> 0): stability needs R''(r) < 0
    d2 = (12.0 * c4, 6.0 * c3, 2.0 * c2)
    ok &= np.where(wide, True, _polyval(d2, rp) < 0.0)
    return ok


def apoapsis_state(a, ra, phi, E, Lz, Q):
    """Cartesian Kerr-Schild 8-vector at apoapsis on the equator, moving 'upward' (u^theta < 0).

    Textbook BL first integrals at theta = pi/2 (rho^2 = r^2), T = E (r^2+a^2) - a Lz:
      u^t = [-a (aE - Lz) + (r^2+a^2) T / Delta] / r^2,  u^phi = [-(aE - Lz) + a T / Delta] / r^2,
      u^r = 0 (turning point), u^theta = -sqrt(Q) / r^2.
    With u^r = 0 the BL and spherical-KS components coincide (the charts differ by functions of r
    only) and x + i y = (r + i a) e^{i phi}, z = 0."""
    r = ra
    delta = r * r - 2.0 * r + a * a
    T = E * (r * r + a * a) - a * Lz
    ut = (-a * (a * E - Lz) + (r * r + a * a) * T / delta) / (r * r)
    uphi = (-(a * E - Lz) + a * T / delta) / (r * r)
    uth = -np.sqrt(np.maximum(Q, 0.0)) / (r * r)
    x = r * np.cos(phi) - a * np.sin(phi)
    y = r * np.sin(phi) + a * np.cos(phi)
    out = np.zeros(r.shape + (8,))
    out[..., 1] = x
    out[..., 2] = y
    out[..., 4] = ut
    out[..., 5] = -y * uphi
    out[..., 6] = x * uphi
    out[..., 7] = -r * uth
    return out


def cfg4_ensemble(n: int, seed: int = 7062, a: float = 0.7, p_range=(8.0, 50.0), e_range=(0.0, 0.8),
                  max_attempts: int = 64):
    """n bound time-like Kerr orbits: p ~ U[p_range], e ~ U[e_range], cos iota ~ U[-1,1], phi ~ U[0,2pi),
    rejection-sampled so that every particle is bound (the stated box is not: the retrograde ISCO at
    a = 0.7 is 8.14 M > 8 M).  Draw t of particle k uses counters 4 (t n + k) + {0,1,2,3}.
    Returns (xu8[n,8], meta) with meta = dict(E, Lz, Q, p, e, cosi, phi, attempts, acceptance)."""
    todo = np.arange(n, dtype=np.uint64)
    cols = {k: np.zeros(n) for k in ("E", "Lz", "Q", "p", "e", "cosi", "phi")}
    attempts = np.zeros(n, dtype=np.int32)
    xu8 = np.zeros((n, 8))
    drawn = accepted = 0
    for t in range(max_attempts):
        if todo.size == 0:
            break
        base = (np.uint64(t) * np.uint64(n) + todo) * np.uint64(4)
        u = [splitmix64_uniform(seed, base + np.uint64(j)) for j in range(4)]
        p = p_range[0] + (p_range[1] - p_range[0]) * u[0]
        e = e_range[0] + (e_range[1] - e_range[0]) * u[1]
        cosi = -1.0 + 2.0 * u[2]
        phi = 2.0 * math.pi * u[3]
        E, Lz, Q, ok = solve_orbit_constants(a, p, e, cosi)
        rp, ra = p / (1.0 + e), p / (1.0 - e)
        ok &= orbit_is_bound(a, E, Lz, Q, rp, ra)
        idx = todo[ok].astype(np.int64)
        xu8[idx] = apoapsis_state(a, ra[ok], phi[ok], E[ok], Lz[ok], Q[ok])
        for key, val in (("E", E), ("Lz", Lz), ("Q", Q), ("p", p), ("e", e), ("cosi", cosi), ("phi", phi)):
            cols[key][idx] = val[ok]
        attempts[idx] = t + 1
        drawn += todo.size
        accepted += int(ok.sum())
        todo = todo[~ok]
    if todo.size:
        raise RuntimeError("cfg4_ensemble: %d particles never accepted" % todo.size)
    meta = dict(cols)
    meta["attempts"] = attempts
    meta["acceptance"] = accepted / max(drawn, 1)
    return xu8, meta
