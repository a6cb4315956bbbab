"""Exact-rational brute force straight from the definitions, for tiny inputs only.

Independent of oracle/ and of the CUDA path: pure Python integers and Fractions, all
grain triples, no cells.  The point-line distance is written the *other* way round from
the oracle's cross product - projection onto the line, dist^2 = |v|^2 - (v.d)^2/|d|^2
(Lagrange's identity makes the two equal) - so a dropped term, a wrong sign or a
transposed operand in either shows up as a disagreement.

Definitions restated from SURVEY.md 8(c) O2..O7 (Fig. 4).
"""
from fractions import Fraction


def _k(g, row):
    x, y, z = g
    return (z, x + y, min(x, y), x, row)


def track_view_exact(grains, params):
    """grains: list of (x,y,z) ints (row = position).  Returns dict with seeds, candidates, tracks."""
    n = len(grains)
    smin2 = params["sep_min_q"] ** 2
    smax2 = params["sep_max_q"] ** 2
    r2 = params["tube_r2_q"]
    nmin = params["min_grains"]
    ext = params.get("tube_ext_q", -1)
    seeds = {}      # (a,b) -> (n_tube, D2, tube set)
    for a in range(n):
        ax, ay, az = grains[a]
        for b in range(a + 1, n):
            d = (grains[b][0] - ax, grains[b][1] - ay, grains[b][2] - az)
            D2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2]
            if not (smin2 <= D2 < smax2):
                continue
            tube = []
            for p in range(n):
                v = (grains[p][0] - ax, grains[p][1] - ay, grains[p][2] - az)
                vv = v[0] * v[0] + v[1] * v[1] + v[2] * v[2]
                vd = v[0] * d[0] + v[1] * d[1] + v[2] * d[2]
                dist2 = Fraction(vv) - Fraction(vd * vd, D2)      # squared distance to the infinite line
                if dist2 > r2:
                    continue
                if ext >= 0:
                    # bounded tube: the foot of P, lam = (v.d)/D2 in units of the seed length,
                    # must lie in [-ext/|d|, 1 + ext/|d|]; beyond an end the overshoot is compared through its square
                    lam = Fraction(vd, D2)
                    over = -lam if lam < 0 else (lam - 1 if lam > 1 else Fraction(0))
                    if over * over * D2 > ext * ext:
                        continue
                tube.append(p)
            seeds[(a, b)] = (len(tube), D2, tube)
    cands = {ab: s for ab, s in seeds.items() if s[0] >= nmin}

    def rank(ab):   # smaller = better: larger n_tube, larger D2, smaller kmin, smaller kmax
        a, b = ab
        ka, kb = _k(grains[a], a), _k(grains[b], b)
        return (-cands[ab][0], -cands[ab][1], min(ka, kb), max(ka, kb))

    owner = {}
    for g in range(n):          # by definition: scan ALL candidates for every grain
        holders = [ab for ab, s in cands.items() if g in s[2]]
        if holders:
            owner[g] = min(holders, key=rank)
    members = {}
    for g, ab in owner.items():
        members.setdefault(ab, []).append(g)
    tracks = [ab for ab, m in members.items() if len(m) >= nmin]
    tracks.sort(key=rank)
    out = []
    for ab in tracks:
        out.append(dict(seed_a=ab[0], seed_b=ab[1], n_tube=cands[ab][0], seed_d2=cands[ab][1],
                        members=sorted(members[ab])))
    return dict(seeds={ab: s[0] for ab, s in seeds.items()}, n_candidates=len(cands), tracks=out)


def fit_exact(points):
    """OLS of the two minor coordinates on the dominant axis with exact rationals."""
    n = len(points)
    ext = [max(p[i] for p in points) - min(p[i] for p in points) for i in range(3)]
    if ext[2] >= ext[0] and ext[2] >= ext[1]:
        u, v, w = 2, 0, 1
    elif ext[0] >= ext[1]:
        u, v, w = 0, 1, 2
    else:
        u, v, w = 1, 0, 2
    mu = Fraction(sum(p[u] for p in points), n)
    out = dict(axis=u, n=n, u_min=min(p[u] for p in points), u_max=max(p[u] for p in points))
    var = sum((p[u] - mu) ** 2 for p in points)
    sl, ic = [], []
    for m in (v, w):
        mm = Fraction(sum(p[m] for p in points), n)
        if var == 0:
            s = Fraction(0)
        else:
            s = sum((p[u] - mu) * (p[m] - mm) for p in points) / var     # cov/var form, not the sums form
        sl.append(s); ic.append(mm - s * mu)
    out["slope"] = sl; out["icpt"] = ic; out["degenerate"] = (var == 0)
    return out
