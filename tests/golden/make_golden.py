"""Writes the stored expected values of tests/golden/ from the paper's printed formulas alone.

It imports neither the oracle nor the CUDA package: the values are what the formulas of
/root/reference/PAPER.md give when typed out in plain Python (lattice sums in float arithmetic with
math.fsum, the Tillotson value in 50-digit decimal arithmetic).  Run `python tests/golden/make_golden.py`
to regenerate lattice_sums.txt and tillotson.txt; `--check` compares with the files instead.
"""
import itertools
import math
import os
import sys
from decimal import Decimal, getcontext

HERE = os.path.dirname(os.path.abspath(__file__))


def s_norm(D):                      # PAPER.md:221 (eq. 26)
    return {1: 4.0 / 3.0, 2: 40.0 / (7.0 * math.pi), 3: 8.0 / math.pi}[D]


def W(D, r, h):                     # PAPER.md:217 (eq. 25): support r <= h
    q = r / h
    if q < 0.5:
        f = 6 * q ** 3 - 6 * q ** 2 + 1
    elif q <= 1.0:
        f = 2 * (1 - q) ** 3
    else:
        f = 0.0
    return s_norm(D) / h ** D * f


def dW(D, r, h):                    # PAPER.md:226 (eq. 27)
    q = r / h
    if q < 0.5:
        f = 3 * q ** 2 - 2 * q
    elif q <= 1.0:
        f = -(1 - q) ** 2
    else:
        f = 0.0
    return 6 * s_norm(D) / h ** (D + 1) * f


def lattice(D, dx=1.0):
    """Interior particle of an infinite lattice of spacing dx, h = 2.6 dx: partner count, density sum of
    eq. 28 with the self term (in units of m / dx^D) and the xx entry of eq. 44's moment matrix
    N = sum_b V_b (x_b - x_a) (x) grad_a W_ab with V_b = dx^D."""
    h = 2.6 * dx
    count, dens, mom = 0, [W(D, 0.0, h) * dx ** D], []
    for nvec in itertools.product(range(-3, 4), repeat=D):
        r = math.sqrt(sum(c * c for c in nvec)) * dx
        if r == 0.0 or not r < h:
            continue
        count += 1
        dens.append(W(D, r, h) * dx ** D)
        # x_b - x_a = n dx;  grad_a W = dW/dr (x_a - x_b)/r
        mom.append(dx ** D * (nvec[0] * dx) * dW(D, r, h) * (-nvec[0] * dx) / r)
    return count, math.fsum(dens), math.fsum(mom)


def tillotson_eq15(m, rho, u):      # PAPER.md:132 (eq. 15), 50 digits
    getcontext().prec = 50
    D = Decimal
    rho0, a, b, A, E0, al, be = (D(m[k]) for k in ("rho0", "a", "b", "A", "E0", "alpha", "beta"))
    rho, u = D(rho), D(u)
    eta = rho / rho0
    z = rho0 / rho - 1
    return float(a * rho * u + (b * rho * u / (1 + u / (E0 * eta * eta)) + A * (eta - 1) * (-be * z).exp())
                 * (-al * z * z).exp())


# basalt: BASELINE.json configs[3] and PAPER.md:615 (Table 1: E_iv, E_cv)
BASALT = dict(rho0=2860.0, A=26.7e9, B=26.7e9, E0=487e6, a=0.5, b=1.5, alpha=5.0, beta=5.0, Ecv=18.2e6)


def contents():
    c2, d2, m2 = lattice(2)
    c3, d3, m3 = lattice(3)
    lat = f"""# Closed-form lattice sums for the cubic B-spline of PAPER.md:217-230 (eqs. 25-27) with
# h = 2.6 dx on an infinite square / cubic lattice of spacing dx (SURVEY.md section 4,
# computed there from the plain lattice sum  sum_n W(|n| dx; 2.6 dx) dx^D  over integer
# vectors n with |n|^2 <= 6, and  N00 = sum_n dx^D n_x dx dW/dx_a  for eq. 44's matrix).
# Written by tests/golden/make_golden.py (plain Python from the printed formulas; no oracle call).
# key value
neighbours_2d {c2}
neighbours_3d {c3}
density_2d {d2!r}
density_3d {d3!r}
moment00_2d {m2!r}
moment00_3d {m3!r}
# Normalisation constants printed in the paper, PAPER.md:221 (eq. 26)
s_1d {s_norm(1)!r}
s_2d {s_norm(2)!r}
s_3d {s_norm(3)!r}
"""
    p = tillotson_eq15(BASALT, 0.9 * BASALT["rho0"], 2.0 * BASALT["Ecv"])
    til = f"""# Tillotson equation of state, expanded and hot branch, PAPER.md:132 (eq. 15), basalt parameters of
# BASELINE.json configs[3] / PAPER.md:615 (Table 1), at eta = rho/rho0 = 0.9 and u = 2 E_cv.
# Written by tests/golden/make_golden.py in 50-digit decimal arithmetic from the printed formula.
# key value
basalt_eq15_eta0.9_u2Ecv {p!r}
"""
    return {"lattice_sums.txt": lat, "tillotson.txt": til}


def _values(text):
    return {l.split()[0]: float(l.split()[1]) for l in text.splitlines() if l.strip() and not l.startswith("#")}


if __name__ == "__main__":
    bad = 0
    for name, text in contents().items():
        path = os.path.join(HERE, name)
        if "--check" in sys.argv:
            have = _values(open(path).read())
            for k, v in _values(text).items():
                if not math.isclose(have[k], v, rel_tol=2e-15, abs_tol=0):
                    print(f"{name}: {k} stored {have[k]!r} recomputed {v!r}")
                    bad += 1
        else:
            with open(path, "w") as fh:
                fh.write(text)
            print("wrote", path)
    sys.exit(1 if bad else 0)
