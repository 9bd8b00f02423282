"""Closed-form / exact reference solutions used to pin the oracle.  Independent of oracle/ and of
the CUDA path: plain numpy written from the relations in SURVEY.md section 8(c) (O9, 'Sod relations')."""
import math
from fractions import Fraction

import numpy as np

CS = 1.0 / math.sqrt(3.0)


# ------------------------------------------------------------------ exact relativistic Sod tube
def _v_rarefaction(e, eL):
    x = (e / eL) ** (math.sqrt(3.0) / 2.0)
    return (1.0 - x) / (1.0 + x)


def _v_shock(e, eR):
    return math.sqrt(3.0) * (e - eR) / math.sqrt((3.0 * eR + e) * (3.0 * e + eR))


def sod_star(eL=10.0, nL=1.0, eR=1.0, nR=0.1):
    lo, hi = eR, eL
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if _v_rarefaction(mid, eL) - _v_shock(mid, eR) > 0.0:
            lo = mid
        else:
            hi = mid
    es = 0.5 * (lo + hi)
    vs = _v_shock(es, eR)
    Vs = math.sqrt((3.0 * es + eR) / (3.0 * (3.0 * eR + es)))
    vprime = 1.0 / (3.0 * Vs)          # downstream speed in the shock frame
    gam = lambda v: 1.0 / math.sqrt(1.0 - v * v)
    nsR = nR * gam(Vs) * Vs / (gam(vprime) * vprime)
    nsL = nL * (es / eL) ** 0.75
    tail = (vs - CS) / (1.0 - vs * CS)
    return dict(e_star=es, p_star=es / 3.0, v_star=vs, shock_speed=Vs, rar_head=-CS, rar_tail=tail,
                n_star_left=nsL, n_star_right=nsR)


def sod_exact(x, t, eL=10.0, nL=1.0, eR=1.0, nR=0.1):
    """e, n, v at positions x (diaphragm at 0) and time t."""
    s = sod_star(eL, nL, eR, nR)
    xi = np.asarray(x, dtype=float) / t
    e = np.empty_like(xi); n = np.empty_like(xi); v = np.empty_like(xi)
    left = xi < s["rar_head"]
    fan = (~left) & (xi < s["rar_tail"])
    starL = (~left) & (~fan) & (xi < s["v_star"])
    starR = (xi >= s["v_star"]) & (xi < s["shock_speed"])
    right = xi >= s["shock_speed"]
    e[left], n[left], v[left] = eL, nL, 0.0
    vf = (xi[fan] + CS) / (1.0 + xi[fan] * CS)
    ef = eL * ((1.0 - vf) / (1.0 + vf)) ** (2.0 / math.sqrt(3.0))
    e[fan], v[fan], n[fan] = ef, vf, nL * (ef / eL) ** 0.75
    e[starL], n[starL], v[starL] = s["e_star"], s["n_star_left"], s["v_star"]
    e[starR], n[starR], v[starR] = s["e_star"], s["n_star_right"], s["v_star"]
    e[right], n[right], v[right] = eR, nR, 0.0
    return e, n, v


# ------------------------------------------------------------------ WENO from its definition
def _solve(A, b):
    """Gauss elimination in exact rationals; A is a list of rows."""
    n = len(A)
    M = [list(map(Fraction, A[i])) + [Fraction(b[i])] for i in range(n)]
    for c in range(n):
        piv = next(r for r in range(c, n) if M[r][c] != 0)
        M[c], M[piv] = M[piv], M[c]
        M[c] = [x / M[c][c] for x in M[c]]
        for r in range(n):
            if r != c and M[r][c] != 0:
                M[r] = [x - M[r][c] * y for x, y in zip(M[r], M[c])]
    return [M[i][n] for i in range(n)]


def _poly_from_averages(cells, f):
    """Coefficients c_m (lowest first) of the polynomial whose average over each unit cell
    [j-1/2, j+1/2], j in `cells`, is f_j."""
    k = len(cells)
    A = [[(Fraction(2 * j + 1, 2) ** (m + 1) - Fraction(2 * j - 1, 2) ** (m + 1)) / (m + 1) for m in range(k)]
         for j in cells]
    return _solve(A, f)


def _peval(c, x):
    return sum(cm * Fraction(x) ** m for m, cm in enumerate(c))


def _pderiv(c):
    return [m * cm for m, cm in enumerate(c)][1:]


def _pmul(a, b):
    out = [Fraction(0)] * (len(a) + len(b) - 1)
    for i, x in enumerate(a):
        for j, y in enumerate(b):
            out[i + j] += x * y
    return out


def _pint(c, lo, hi):
    return sum(cm * (Fraction(hi) ** (m + 1) - Fraction(lo) ** (m + 1)) / (m + 1) for m, cm in enumerate(c))


def weno_exact(f, eps):
    """FD-WENO value at i+1/2 from the definition (Jiang-Shu / Balsara-Shu), exact rationals.
    f has 2r-1 entries f_{i-r+1..i+r-1}.  Candidate k uses cells i-r+1+k .. i+k; q_k = p_k(1/2);
    beta_k = sum_{l=1}^{r-1} int_{-1/2}^{1/2} (d^l p_k/dx^l)^2 dx (dx = 1); d_k = the linear weights that
    reproduce the (2r-1)-cell polynomial; alpha_k = d_k/(eps+beta_k)^2."""
    f = [Fraction(x) for x in f]
    r = (len(f) + 1) // 2
    allc = list(range(-r + 1, r))
    q, beta = [], []
    for k in range(r):
        cells = allc[k:k + r]
        c = _poly_from_averages(cells, f[k:k + r])
        q.append(_peval(c, Fraction(1, 2)))
        b = Fraction(0)
        d = c
        for _ in range(1, r):
            d = _pderiv(d)
            b += _pint(_pmul(d, d), Fraction(-1, 2), Fraction(1, 2))
        beta.append(b)
    # linear weights: match the full-stencil reconstruction as a linear functional of f
    rows, rhs = [], []
    for j in range(2 * r - 1):
        unit = [Fraction(1 if m == j else 0) for m in range(2 * r - 1)]
        full = _peval(_poly_from_averages(allc, unit), Fraction(1, 2))
        row = []
        for k in range(r):
            if k <= j < k + r:
                row.append(_peval(_poly_from_averages(allc[k:k + r], unit[k:k + r]), Fraction(1, 2)))
            else:
                row.append(Fraction(0))
        rows.append(row); rhs.append(full)
    d = _solve(rows[:r], rhs[:r])
    for row, b in zip(rows, rhs):      # the over-determined system must be consistent
        assert sum(x * y for x, y in zip(row, d)) == b
    eps = Fraction(eps)
    al = [dk / (eps + bk) ** 2 for dk, bk in zip(d, beta)]
    s = sum(al)
    return sum(a / s * qk for a, qk in zip(al, q)), dict(q=q, beta=beta, d=d)
