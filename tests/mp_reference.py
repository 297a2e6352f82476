"""50-digit mpmath evaluations used to pin the CPU oracle on tiny inputs.

Written from the DEFINITIONS (DESIGN.md readings), independently of
oracle/mopal_oracle.c: different language, different precision, and for the
drift a different formulation (classical elements + Kepler's equation instead of
universal variables).  Test-only.
"""
import mpmath as mp

mp.mp.dps = 50


def K_mp(s, rc):
    """changeover weight, reading A-1/A-4: quintic smoothstep on [0.1 rc, rc]."""
    if rc == 0 or s >= rc:
        return mp.mpf(1)
    if s <= rc / 10:
        return mp.mpf(0)
    q = (s - rc / 10) / (rc * 9 / 10)
    return 10 * q**3 - 15 * q**4 + 6 * q**5


def accel_mp(gm, x, rcrit):
    nb = len(gm)
    X = [[mp.mpf(float(x[c][b])) for c in range(3)] for b in range(nb)]
    out, S = [], []
    for i in range(nb):
        a = [mp.mpf(0)] * 3
        s_ = [mp.mpf(0)] * 3
        for j in range(nb):
            if j == i:
                continue
            d = [X[j][c] - X[i][c] for c in range(3)]
            r = mp.sqrt(sum(t * t for t in d))
            if r == 0:
                continue
            rc = max(mp.mpf(float(rcrit[i])), mp.mpf(float(rcrit[j])))
            w = mp.mpf(float(gm[j])) * K_mp(r, rc) / r**3
            a = [a[c] + w * d[c] for c in range(3)]
            s_ = [s_[c] + abs(w * d[c]) for c in range(3)]
        out.append(a)
        S.append(s_)
    return out, S


def hermite_extremes_mp(p0, p1, w0, w1, h):
    """extremes over tau in [0,1] of the cubic Hermite interpolant (reading B-a),
    found by polynomial root finding rather than the oracle's closed form."""
    p0, p1, w0, w1, h = map(mp.mpf, (p0, p1, w0, w1, h))
    k1 = h * w0
    k2 = 3 * (p1 - p0) - h * (2 * w0 + w1)
    k3 = -2 * (p1 - p0) + h * (w0 + w1)
    cand = [p0, p1]
    if w0 * w1 < 0:
        coeffs = [3 * k3, 2 * k2, k1]
        while coeffs and coeffs[0] == 0:
            coeffs = coeffs[1:]
        if len(coeffs) > 1:
            for r in mp.polyroots(coeffs, maxsteps=200, extraprec=200):
                if mp.im(r) == 0 or abs(mp.im(r)) < mp.mpf(10) ** -40:
                    t = mp.re(r)
                    if 0 < t < 1:
                        cand.append(((k3 * t + k2) * t + k1) * t + p0)
    return min(cand), max(cand)


def d2min_mp(h, X0i, V0i, X1i, V1i, X0j, V0j, X1j, V1j):
    """reading B-d by root finding on the derivative of the cubic of d^2."""
    f = lambda a: [mp.mpf(float(t)) for t in a]
    X0i, V0i, X1i, V1i, X0j, V0j, X1j, V1j = map(f, (X0i, V0i, X1i, V1i, X0j, V0j, X1j, V1j))
    h = mp.mpf(float(h))
    D0 = [a - b for a, b in zip(X0i, X0j)]
    D1 = [a - b for a, b in zip(X1i, X1j)]
    U0 = [a - b for a, b in zip(V0i, V0j)]
    U1 = [a - b for a, b in zip(V1i, V1j)]
    d0 = sum(t * t for t in D0)
    d1 = sum(t * t for t in D1)
    d0t = 2 * sum(a * b for a, b in zip(D0, U0))
    d1t = 2 * sum(a * b for a, b in zip(D1, U1))
    if d0t * h <= 0 and d1t * h >= 0:
        c1 = h * d0t
        c2 = 3 * (d1 - d0) - h * (2 * d0t + d1t)
        c3 = -2 * (d1 - d0) + h * (d0t + d1t)
        cub = lambda t: ((c3 * t + c2) * t + c1) * t + d0
        # the stationary point where the derivative goes from <=0 to >=0
        best = min(d0, d1)
        coeffs = [3 * c3, 2 * c2, c1]
        while coeffs and coeffs[0] == 0:
            coeffs = coeffs[1:]
        if len(coeffs) > 1:
            for r in mp.polyroots(coeffs, maxsteps=500, extraprec=400):
                if abs(mp.im(r)) < mp.mpf(10) ** -35:
                    t = min(max(mp.re(r), 0), 1)
                    second = 6 * c3 * t + 2 * c2
                    if second >= 0:
                        best = min(best, max(cub(t), 0))
        return best, d0, d1
    return min(d0, d1), d0, d1


def kepler_elements_propagate_mp(mu, dt, x, v):
    """Two-body propagation via classical elements and Kepler's equation
    (elliptic orbits only)."""
    mu = mp.mpf(float(mu)); dt = mp.mpf(float(dt))
    r0 = [mp.mpf(float(t)) for t in x]
    v0 = [mp.mpf(float(t)) for t in v]
    dot = lambda a, b: sum(p * q for p, q in zip(a, b))
    cross = lambda a, b: [a[1] * b[2] - a[2] * b[1], a[2] * b[0] - a[0] * b[2], a[0] * b[1] - a[1] * b[0]]
    r = mp.sqrt(dot(r0, r0))
    v2 = dot(v0, v0)
    a = 1 / (2 / r - v2 / mu)
    assert a > 0
    hvec = cross(r0, v0)
    evec = [c / mu - p / r for c, p in zip(cross(v0, hvec), r0)]
    e = mp.sqrt(dot(evec, evec))
    n = mp.sqrt(mu / a**3)
    # eccentric anomaly at t0 from r = a(1 - e cos E), r.v = sqrt(mu a) e sin E
    ecosE = 1 - r / a
    esinE = dot(r0, v0) / mp.sqrt(mu * a)
    E0 = mp.atan2(esinE, ecosE)
    M0 = E0 - esinE
    M1 = M0 + n * dt
    E1 = mp.findroot(lambda E: E - e * mp.sin(E) - M1, M1 + e * mp.sin(M1), tol=mp.mpf(10) ** -45, maxsteps=200)
    dE = E1 - E0
    # Gauss f, g in terms of the eccentric anomaly difference
    f = 1 - a / r * (1 - mp.cos(dE))
    g = dt - (dE - mp.sin(dE)) / n
    r1 = a * (1 - e * mp.cos(E1))
    fd = -mp.sqrt(mu * a) / (r * r1) * mp.sin(dE)
    gd = 1 - a / r1 * (1 - mp.cos(dE))
    xn = [f * p + g * q for p, q in zip(r0, v0)]
    vn = [fd * p + gd * q for p, q in zip(r0, v0)]
    return xn, vn
