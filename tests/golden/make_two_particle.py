"""Provenance of tests/golden/two_particle.txt: re-evaluates its six rows in 40-digit arithmetic.

Independent of oracle/ and of the CUDA path (imports neither): it is the definition typed out once
more with mpmath -- Eq. 3 (reading G1: second term of the first branch is
38.4 r^3/h^5) and the literal Eq. 8 window  |r_z - n L| < N_cut L  on the RAW r_z (PAPER.md:85-90,
no nearest-image wrap, no sign rule), which is a different route to the image set from the one the
oracle takes (wrap, then n = -N_cut+1 .. N_cut-1 plus one sign-selected end image).

    python tests/golden/make_two_particle.py            # prints the table
    python tests/golden/make_two_particle.py --check    # compares with two_particle.txt (1e-15 relative)
"""
import os
import sys

from mpmath import mp, mpf, sqrt

mp.dps = 40

ROWS = [  # r_x r_y r_z h L N_cut   (h = h_i + h_j, the spline support of the pair; G = m_j = 1)
    ("1", "0", "0", "1", "100", 1),
    ("0.25", "0", "0", "1", "100", 1),
    ("0.3", "0", "0.1", "1", "100", 5),
    ("0.6", "0.3", "-0.2", "1", "100", 3),
    ("3", "4", "20", "1", "100", 5),
    ("0.2", "0.1", "49.9", "0.4", "100", 2),
]


def spline_F(r, h):
    """Eq. 3: force magnitude of the M4 spline-softened unit mass, support h."""
    if r >= h:
        return 1 / r**2
    if r >= h / 2:
        return (-mpf(32) / 3 * r**4 / h**6 + mpf("38.4") * r**3 / h**5 - 48 * r**2 / h**4
                + mpf(64) / 3 * r / h**3 - 1 / (15 * r**2))
    return 32 * r**4 / h**6 - mpf("38.4") * r**3 / h**5 + mpf(32) / 3 * r / h**3


def accel(rx, ry, rz, h, L, ncut):
    """Eq. 8 on the raw separation: every integer n with |r_z - n L| < N_cut L (strict)."""
    g = [mpf(0)] * 3
    for n in range(-2 * ncut - 2, 2 * ncut + 3):
        d = rz - n * L
        if not abs(d) < ncut * L:
            continue
        s = sqrt(rx**2 + ry**2 + d**2)
        if s == 0:
            continue
        w = spline_F(s, h) / s
        g = [g[0] - w * rx, g[1] - w * ry, g[2] - w * d]
    return g


def table():
    out = []
    for rx, ry, rz, h, L, nc in ROWS:
        g = accel(mpf(rx), mpf(ry), mpf(rz), mpf(h), mpf(L), nc)
        out.append(((rx, ry, rz, h, L, nc), g))
    return out


def main():
    rows = table()
    if "--check" not in sys.argv:
        for (rx, ry, rz, h, L, nc), g in rows:
            print(rx, ry, rz, h, L, nc, *[mp.nstr(v, 20) for v in g])
        return 0
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "two_particle.txt")
    stored = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    assert len(stored) == len(rows)
    worst = mpf(0)
    for cols, (_, g) in zip(stored, rows):
        for a, b in zip(cols[6:9], g):
            a = mpf(a)
            scale = max(abs(b), mpf("1e-300"))
            err = abs(a - b) / scale if b != 0 else abs(a)
            worst = max(worst, err)
    print("max relative difference to two_particle.txt:", mp.nstr(worst, 3))
    return 0 if worst < mpf("1e-15") else 1


if __name__ == "__main__":
    sys.exit(main())
