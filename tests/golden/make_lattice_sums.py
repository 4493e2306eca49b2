#!/usr/bin/env python
"""Generator of tests/golden/lattice_sums.txt -- pure Python, imports NOTHING from oracle/ or the CUDA package.

    python tests/golden/make_lattice_sums.py            # prints the table (key value)
    python tests/golden/make_lattice_sums.py --check    # compares with the committed file, exit 1 on a mismatch

Every number is what the mathematics fixes for a static lattice (SURVEY.md 8(c) pins P2, P6, P7, P8): closed
forms of the shifted-force pair functions ("truncation plus shift of the pair force", i.e. a linear
term in the potential) written out here once more in plain Python floats, summed over INTEGER lattice vectors.
Nothing here knows about particles, boxes, neighbour lists or minimum images.
"""
from __future__ import annotations

import itertools
import math
import os
import sys


def lj(r, eps=1.0, sig=1.0):
    """u = 4 eps [(s/r)^12 - (s/r)^6], f = -du/dr = (24 eps / r) [2 (s/r)^12 - (s/r)^6]."""
    s6 = (sig / r) ** 6
    return 4.0 * eps * (s6 * s6 - s6), 24.0 * eps * (2.0 * s6 * s6 - s6) / r


def coulomb(r, qq):
    return qq / r, qq / (r * r)


def cut(raw, r, rc, method):
    """method 0 shifted force: u(r) - u(rc) + (r - rc) f(rc), f(r) - f(rc); 1 shifted potential; 2 no shift."""
    if r >= rc:
        return 0.0, 0.0
    u, f = raw(r)
    uc, fc = raw(rc)
    if method == 0:
        return u - uc + (r - rc) * fc, f - fc
    if method == 1:
        return u - uc, f
    return u, f


def shells(vectors, a, radii):
    """Squared integer norms -> distances; returns [(distance, integer vector)], and the counts inside each radius."""
    out = [(a * math.sqrt(n2), v) for n2, v in vectors]
    counts = [sum(1 for d, _ in out if d < R) for R in radii]
    return out, counts


def fcc_vectors(m=6):
    """fcc lattice vectors in units of a/2: integer (i, j, k) with i + j + k even, distance (a/2) sqrt(i^2+j^2+k^2)."""
    for i, j, k in itertools.product(range(-m, m + 1), repeat=3):
        if (i + j + k) % 2 == 0 and (i, j, k) != (0, 0, 0):
            yield (i * i + j * j + k * k) / 4.0, (i, j, k)


def sc_vectors(m=6):
    for i, j, k in itertools.product(range(-m, m + 1), repeat=3):
        if (i, j, k) != (0, 0, 0):
            yield float(i * i + j * j + k * k), (i, j, k)


def bisect_root(fn, lo, hi):
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if fn(mid) > 0:
            lo = mid
        else:
            hi = mid
    return lo


def table():
    T = []
    uc, fc = lj(2.5)
    T += [("sf_lj_u_rc", uc), ("sf_lj_f_rc", fc)]
    r0 = 2.0 ** (1.0 / 6.0)
    T.append(("sf_lj_u_at_2p16", cut(lj, r0, 2.5, 0)[0]))
    rmin = bisect_root(lambda r: cut(lj, r, 2.5, 0)[1], 1.0, 1.3)
    T += [("sf_lj_rmin", rmin), ("sf_lj_umin", cut(lj, rmin, 2.5, 0)[0])]
    # P6: fcc at density 0.8442
    a = (4.0 / 0.8442) ** (1.0 / 3.0)
    sh, (n_rc, n_list) = shells(fcc_vectors(), a, [2.5, 2.8])
    U = sum(cut(lj, d, 2.5, 0)[0] for d, _ in sh)
    Wv = sum(d * cut(lj, d, 2.5, 0)[1] for d, _ in sh)
    T += [("fcc_a", a), ("fcc_u_per_n", 0.5 * U), ("fcc_w_per_n", 0.5 * Wv), ("fcc_n_inside_rc", n_rc),
          ("fcc_n_list", n_list)]
    # P7: rock salt (simple cubic sites, charge (-1)^(i+j+k)) at density 0.5
    a = 0.5 ** (-1.0 / 3.0)
    sh, (n25, n40, n43) = shells(sc_vectors(), a, [2.5, 4.0, 4.3])
    ulj = sum(cut(lj, d, 2.5, 0)[0] for d, _ in sh)
    wlj = sum(d * cut(lj, d, 2.5, 0)[1] for d, _ in sh)
    ucl = wcl = 0.0
    for d, v in sh:
        qq = 1.0 if sum(v) % 2 == 0 else -1.0
        u, f = cut(lambda r: coulomb(r, qq), d, 4.0, 0)
        ucl += u
        wcl += d * f
    T += [("rocksalt_a", a), ("rocksalt_u_coul_per_n", 0.5 * ucl), ("rocksalt_u_lj_per_n", 0.5 * ulj),
          ("rocksalt_u_per_n", 0.5 * (ucl + ulj)), ("rocksalt_w_per_n", 0.5 * (wcl + wlj)),
          ("rocksalt_n_inside_2p5", n25), ("rocksalt_n_inside_4p0", n40), ("rocksalt_n_list", n43)]
    # P8: simple-cubic sites of the Kob-Andersen start, a = 1.2^(-1/3), inside the three LIST radii (rc + 0.3)
    a = 1.2 ** (-1.0 / 3.0)
    _, (aa, ab, bb) = shells(sc_vectors(), a, [2.5 + 0.3, 2.0 + 0.3, 2.2 + 0.3])
    T += [("ka_sc_sites_aa", aa), ("ka_sc_sites_ab", ab), ("ka_sc_sites_bb", bb)]
    # P6 "for reference": the other two cutoff methods on the same fcc lattice
    a = (4.0 / 0.8442) ** (1.0 / 3.0)
    sh, _ = shells(fcc_vectors(), a, [])
    T += [("fcc_u_per_n_noshift", 0.5 * sum(cut(lj, d, 2.5, 2)[0] for d, _ in sh)),
          ("fcc_u_per_n_shiftedpot", 0.5 * sum(cut(lj, d, 2.5, 1)[0] for d, _ in sh))]
    return T


def committed():
    out = {}
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "lattice_sums.txt")) as fh:
        for line in fh:
            f = line.split("#")[0].split()
            if len(f) == 2:
                out[f[0]] = float(f[1])
    return out


def check(rel=1e-9):
    """Every generated value against the committed file, to the digits the file prints (the statistical pin
    ka_sc_u_per_n_mean is a Monte-Carlo mean over type assignments and is not generated here)."""
    have = committed()
    bad = []
    for k, v in table():
        if k not in have or abs(have[k] - v) > rel * max(1.0, abs(v)):
            bad.append((k, v, have.get(k)))
    return bad


if __name__ == "__main__":
    if "--check" in sys.argv:
        bad = check()
        for k, v, h in bad:
            print("MISMATCH %s generated %.12f file %r" % (k, v, h))
        sys.exit(1 if bad else 0)
    for k, v in table():
        print("%-26s %s" % (k, ("%d" % v) if isinstance(v, int) else ("%.12f" % v)))
