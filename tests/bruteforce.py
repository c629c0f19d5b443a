"""Independent checker for the oracle (pins B1/B2 of SURVEY.md §8(c)).

Written from the SET / PATH forms of D3..D8, not from the oracle's procedure: peaks are the
cells that no neighbour beats, members are found by enumerating descent paths, weights are
exact ``Fraction(Q, S)``.  Different language, different data structures (dict of cells, sets),
exact rational arithmetic; shares nothing with oracle/ or the CUDA path.
"""
from fractions import Fraction
from math import sqrt

NB8 = [(dp, dt) for dt in (-1, 0, 1) for dp in (-1, 0, 1) if (dp, dt) != (0, 0)]


def cheb(a, b):
    return max(abs(a[0] - b[0]), abs(a[1] - b[1]))


def greater(Q, a, b):
    """D3: a beats b.  Cells are (pad, time); key = time*256 + pad, smaller key wins ties."""
    qa, qb = Q.get(a, 0), Q.get(b, 0)
    if qa != qb:
        return qa > qb
    return (a[1] * 256 + a[0]) < (b[1] * 256 + b[0])


def peaks_of(Q, theta):
    """D4 as a set: cells with Q >= theta that beat every one of their 8 neighbours."""
    out = set()
    for c, q in Q.items():
        if q < theta:
            continue
        if all(greater(Q, c, (c[0] + dp, c[1] + dt)) for dp, dt in NB8):
            out.add(c)
    return out


def members_of(Q, peaks, P):
    """D5 path form: c is a member iff a path P=c0..ck=c exists with k<=2, consecutive cells
    8-adjacent, cheb(P,cj)=j, Q(cj) >= Q(cj+1) > 0, and c is not a peak."""
    mem = set()
    ring1 = [(P[0] + dp, P[1] + dt) for dp, dt in NB8]
    for c1 in ring1:
        q1 = Q.get(c1, 0)
        if not (Q[P] >= q1 > 0):
            continue
        if c1 not in peaks:
            mem.add(c1)
        # NB: a ring-1 cell can carry a path even though it cannot itself be a peak (it is
        # adjacent to P), so the "not a peak" test applies to the END of the path only.
        for dp, dt in NB8:
            c2 = (c1[0] + dp, c1[1] + dt)
            if cheb(P, c2) != 2:
                continue
            q2 = Q.get(c2, 0)
            if q1 >= q2 > 0 and c2 not in peaks:
                mem.add(c2)
    return mem


def clusters(Q, theta, npads, tf_time_bins, core=None):
    """All clusters of one (pad x time) map.  Q: {(pad,time): q16>0}.  Returns a list of dicts
    sorted by (time, pad) with exact Fractions for the moments (D6..D8, D10)."""
    Q = {c: q for c, q in Q.items() if q > 0}
    pk = peaks_of(Q, theta)
    res = []
    for P in sorted(pk, key=lambda c: (c[1], c[0])):
        if core is not None and not (core[0] <= P[1] < core[1]):
            continue
        mem = members_of(Q, pk, P)
        W = Fraction(Q[P])
        Mp = Mt = Mpp = Mtt = Fraction(0)
        split = False
        sat = Q[P] == 16368
        for c in mem:
            S = sum(1 for jt in range(-2, 3) for jp in range(-2, 3) if (c[0] + jp, c[1] + jt) in pk)
            assert S >= 1
            w = Fraction(Q[c], S)
            dp, dt = c[0] - P[0], c[1] - P[1]
            W += w
            Mp += w * dp
            Mt += w * dt
            Mpp += w * dp * dp
            Mtt += w * dt * dt
            split |= S >= 2
            sat |= Q[c] == 16368
        flags = 0
        if P[0] < 2 or P[0] >= npads - 2:
            flags |= 1
        if P[1] < 2 or P[1] >= tf_time_bins - 2:
            flags |= 2
        if sat:
            flags |= 4
        if split:
            flags |= 8
        var_p = Mpp / W - (Mp / W) ** 2
        var_t = Mtt / W - (Mt / W) ** 2
        assert var_p >= 0 and var_t >= 0
        res.append(
            dict(pad=P[0], time=P[1], flags=flags, qmax_q16=Q[P], ncells=1 + len(mem),
                 W16=W, qtot=float(W / 16), dpad=float(Mp / W), dtime=float(Mt / W),
                 sigma_pad=sqrt(var_p), sigma_time=sqrt(var_t))
        )
    return res
