"""Independent brute-force statement of the sweep for TINY meshes (pure Python, exact rationals).

Used only by the oracle's pin tests.  It is a different algorithm from oracle/oracle.c: instead of
marching slab by slab with integer crossing tests, it takes each lattice ray as a whole line,
collects every parameter value at which the line meets a cell boundary plane (of any of the three
axes) as an exact Fraction, sorts them, and classifies each open interval by the cell that contains
its midpoint.  Lengths are exact rationals times L.  The physics (eqs. 7-13) is then
applied in plain Python floats along each ray's interval list.

Same reading of the paper as DESIGN.md (dominant-axis lattice, cell-centre offsets, slopes quantised
to 2^-20, zero-length pieces dropped), written separately so that an indexing / sign / ordering
mistake in oracle.c shows up as a disagreement.
"""
from __future__ import annotations

import math
from fractions import Fraction

ONE = 1 << 20


def dir_record(n):
    ab = [abs(float(v)) for v in n]
    a = 0
    for i in (1, 2):
        if ab[i] > ab[a]:
            a = i
    b, c = [i for i in range(3) if i != a]
    Mb = min(ONE, int(round_half_even(ab[b] / ab[a] * ONE)))
    Mc = min(ONE, int(round_half_even(ab[c] / ab[a] * ONE)))
    refl = [float(v) < 0.0 for v in n]
    L = math.sqrt(1.0 + (Mb / ONE) ** 2 + (Mc / ONE) ** 2)
    return a, b, c, refl, Mb, Mc, L


def round_half_even(x):
    f = math.floor(x)
    r = x - f
    if r > 0.5 or (r == 0.5 and f % 2 == 1):
        return f + 1
    return f


def ray_intervals(dims, n, p, q, rays=1):
    """Exact (cell, fraction_of_L) list, in marching order, for lattice ray (p, q) of direction n."""
    a, b, c, refl, Mb, Mc, L = dir_record(n)
    Na, Nb, Nc = dims[a], dims[b], dims[c]
    mb, mc = Fraction(Mb, ONE), Fraction(Mc, ONE)
    # lattice of spacing 1/rays on the plane a = 0 (rays = 1: cell-centre offsets)
    b0, c0 = Fraction(2 * p + 1, 2 * rays), Fraction(2 * q + 1, 2 * rays)
    events = {Fraction(k) for k in range(Na + 1)}
    if Mb:
        lo, hi = math.floor(b0), math.ceil(b0 + mb * Na)
        for g in range(lo, hi + 1):
            s = (Fraction(g) - b0) / mb
            if 0 <= s <= Na:
                events.add(s)
    if Mc:
        lo, hi = math.floor(c0), math.ceil(c0 + mc * Na)
        for g in range(lo, hi + 1):
            s = (Fraction(g) - c0) / mc
            if 0 <= s <= Na:
                events.add(s)
    ev = sorted(events)
    out = []
    for s0, s1 in zip(ev[:-1], ev[1:]):
        if s1 <= s0:
            continue
        mid = (s0 + s1) / 2
        k = math.floor(mid)
        j = math.floor(b0 + mb * mid)
        l = math.floor(c0 + mc * mid)
        if not (0 <= k < Na and 0 <= j < Nb and 0 <= l < Nc):
            continue
        idx = [0, 0, 0]
        idx[a] = Na - 1 - k if refl[a] else k
        idx[b] = Nb - 1 - j if refl[b] else j
        idx[c] = Nc - 1 - l if refl[c] else l
        if not out:
            # entry face: the boundary plane the entry point lies on (edge or corner of two side planes: c)
            if s0 == 0:
                ax = a
            elif c0 + mc * s0 == 0:
                ax = c
            else:
                assert b0 + mb * s0 == 0
                ax = b
            ENTRY_FACE[(tuple(n), p, q, rays)] = 2 * ax + (1 if refl[ax] else 0)
        out.append((tuple(idx), s1 - s0))
    return out, L


ENTRY_FACE = {}


def lattice(dims, n, rays=1):
    a, b, c, refl, Mb, Mc, L = dir_record(n)
    Na, Nb, Nc = dims[a], dims[b], dims[c]
    pmin = -math.ceil(Fraction(Na * Mb, ONE)) - 1
    qmin = -math.ceil(Fraction(Na * Mc, ONE)) - 1
    return [(p, q) for q in range(rays * qmin, rays * Nc) for p in range(rays * pmin, rays * Nb)]


def f_of(x):
    return 1.0 - 0.5 * x if x < 1e-8 else -math.expm1(-x) / x


def sweep(kappa, S, dirs, Ibc=0.0, linear=False, rays=1, Ibc_faces=None):
    """kappa, S: nested [z][y][x] python/numpy arrays (single bin).  Returns dict of per-cell dicts.

    linear=True replaces eq. 7 by the optically thin limit I += kappa*S*ds and f by 1 (pin P6).
    """
    nz, ny, nx = len(kappa), len(kappa[0]), len(kappa[0][0])
    dims = (nx, ny, nz)
    Jin, cnt_tot, per_dir = {}, {}, []
    for n in dirs:
        num, den, cnt, exits = {}, {}, {}, {}
        for (p, q) in lattice(dims, n, rays):
            iv, L = ray_intervals(dims, n, p, q, rays)
            I = float(Ibc)
            if Ibc_faces is not None and iv:
                I = float(Ibc_faces[ENTRY_FACE[(tuple(n), p, q, rays)]])
            chord = 0.0
            for (x, y, z), frac in iv:
                ds = float(frac) * L
                kap, src = float(kappa[z][y][x]), float(S[z][y][x])
                dtau = kap * ds
                cell = (x, y, z)
                if linear:
                    num[cell] = num.get(cell, 0.0) + ds * I
                    I = I + kap * src * ds
                else:
                    num[cell] = num.get(cell, 0.0) + ds * I * f_of(dtau)
                    I = I * math.exp(-dtau) + src * (-math.expm1(-dtau))
                den[cell] = den.get(cell, 0.0) + ds
                cnt[cell] = cnt.get(cell, 0) + 1
                chord += ds
            exits[(p, q)] = (I, chord)
        for cell in den:
            Jin[cell] = Jin.get(cell, 0.0) + num[cell] / den[cell] / len(dirs)
            cnt_tot[cell] = cnt_tot.get(cell, 0) + cnt[cell]
        per_dir.append({"den": den, "cnt": cnt, "exits": exits})
    return {"Jin": Jin, "cnt": cnt_tot, "per_dir": per_dir}
