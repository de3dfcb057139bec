"""T0 oracle: pure-Python, definitional, for tiny maps only.

TEST INFRASTRUCTURE, NOT PRODUCT (see ``oracle/__init__.py``).

Same specification as T1 but formulated differently on
purpose, so that T0 == T1 on exhaustive tiny maps is a real check:

* the map is a dict, not an array (O0);
* the peak test does not compare charges pairwise: all cells of a
  (sector,row) are ranked ONCE by a global sort under the total order of
  O1/Q7 (charge descending, time ascending, pad ascending) and a cell is a
  peak iff its rank is smaller than the rank of each in-range 8-neighbour;
* neighbourhoods and the common-neighbour set of O2 are Python set
  intersections, not index arithmetic;
* O4 uses numpy float32 scalars (each operator rounds once to binary32).
"""
from __future__ import annotations

from itertools import product

import numpy as np

F = np.float32


def n8(c):
    t, p = c
    return {(t + dt, p + dp) for dt, dp in product((-1, 0, 1), repeat=2) if (dt, dp) != (0, 0)}


def build_maps(digits, n_sectors, n_rows, n_time, n_pads):
    """O0.  digits: iterable of (sector,row,pad,time,charge). Returns (maps, bad)."""
    maps = {}
    bad = False
    for (s, r, p, t, q) in digits:
        if s >= n_sectors or r >= n_rows or p >= n_pads[r] or t >= n_time:
            bad = True
            continue
        q = min(q, 1023)
        if q == 0:
            continue
        m = maps.setdefault((s, r), {})
        m[(t, p)] = max(m.get((t, p), 0), q)
    return maps, bad


def peaks_of(m, T, P, thr_peak):
    """O1 by global ranking."""
    cells = [(t, p) for t in range(T) for p in range(P)]
    ranked = sorted(cells, key=lambda c: (-m.get(c, 0), c[0], c[1]))
    rank = {c: i for i, c in enumerate(ranked)}
    pk = set()
    for c in cells:
        if m.get(c, 0) < thr_peak:
            continue
        if all(rank[c] < rank[n] for n in n8(c) if n in rank):
            pk.add(c)
    return pk, rank


def survivors_of(m, pk, rank, noise_eps):
    """O2: single pass against the un-updated peak set."""
    out = set()
    for c in pk:
        qc = m[c]
        dead = False
        for c2 in pk:
            if max(abs(c2[0] - c[0]), abs(c2[1] - c[1])) != 2:
                continue
            if not rank[c2] < rank[c]:
                continue
            common = n8(c) & n8(c2)
            if any(m.get(x, 0) + noise_eps >= qc for x in common):
                dead = True
                break
        if not dead:
            out.add(c)
    return out


def cluster_of(m, T, P, c, s, r, cog_gated=False):
    """O3 + O4 (flags as in O4).  cog_gated = reading Q10' (R7): an outer-ring cell of the
    window counts only if the inner cell between it and the peak holds charge."""
    t_c, p_c = c
    Q = Sp = St = Spp = Stt = 0
    for dt, dp in product(range(-2, 3), repeat=2):
        x = (t_c + dt, p_c + dp)
        if not (0 <= x[0] < T and 0 <= x[1] < P):
            continue
        q = m.get(x, 0)
        if cog_gated and max(abs(dt), abs(dp)) == 2:
            inner = (t_c + max(-1, min(1, dt)), p_c + max(-1, min(1, dp)))
            if m.get(inner, 0) == 0:     # the inner cell is in range whenever the outer one is
                continue
        Q += q
        Sp += q * dp
        St += q * dt
        Spp += q * dp * dp
        Stt += q * dt * dt
    Vp = Q * Spp - Sp * Sp
    Vt = Q * Stt - St * St
    fQ = F(Q)
    pad_mean = F(p_c) + F(Sp) / fQ
    time_mean = F(t_c) + F(St) / fQ
    sigma_pad = np.sqrt(F(Vp)) / fQ
    sigma_time = np.sqrt(F(Vt)) / fQ
    flags = 0
    if p_c < 2 or p_c + 2 >= P:
        flags |= 1
    if t_c < 2 or t_c + 2 >= T:
        flags |= 2
    if m[c] == 1023:
        flags |= 4
    return dict(
        pad_mean=F(pad_mean), time_mean=F(time_mean), sigma_pad=F(sigma_pad), sigma_time=F(sigma_time),
        q_tot=Q, q_max=m[c], time_peak=t_c, pad_peak=p_c, row=r, sector=s, flags=flags, reserved=0,
        sums=(Q, Sp, St, Spp, Stt, Vp, Vt),
    )


def cheb(a, b):
    return max(abs(a[0] - b[0]), abs(a[1] - b[1]))


def cluster_shared_of(m, T, P, c, sv, s, r):
    """O3 + O4 in reading Q10'' (R8): a cell of c's window that also lies in the window of
    partners of c -- survivors at Chebyshev distance exactly 2 from c -- is split by the integer weights
    w_p(x) = (q_p >> 2 cheb(p, x)) + 1; c takes floor(q_x w_c / sum of the weights).  Peak cells are
    never split: c keeps its own in full and takes nothing of a partner's."""
    partners = [p for p in sv if cheb(p, c) == 2]
    t_c, p_c = c
    Q = Sp = St = Spp = Stt = 0
    for dt, dp in product(range(-2, 3), repeat=2):
        x = (t_c + dt, p_c + dp)
        q = m.get(x, 0) if (0 <= x[0] < T and 0 <= x[1] < P) else 0
        if q == 0:
            continue
        if x == c:
            share = q                      # the peak cell is never split
        elif x in partners:
            share = 0                      # nor is a partner's
        else:
            weights = {p: (m[p] >> (2 * cheb(p, x))) + 1 for p in [c] + partners if cheb(p, x) <= 2}
            share = (q * weights[c]) // sum(weights.values())
        Q += share
        Sp += share * dp
        St += share * dt
        Spp += share * dp * dp
        Stt += share * dt * dt
    Vp = Q * Spp - Sp * Sp
    Vt = Q * Stt - St * St
    fQ = F(Q)
    flags = (1 if (p_c < 2 or p_c + 2 >= P) else 0) | (2 if (t_c < 2 or t_c + 2 >= T) else 0) | (4 if m[c] == 1023 else 0)
    return dict(
        pad_mean=F(F(p_c) + F(Sp) / fQ), time_mean=F(F(t_c) + F(St) / fQ), sigma_pad=F(np.sqrt(F(Vp)) / fQ),
        sigma_time=F(np.sqrt(F(Vt)) / fQ), q_tot=Q, q_max=m[c], time_peak=t_c, pad_peak=p_c, row=r, sector=s,
        flags=flags, reserved=0, sums=(Q, Sp, St, Spp, Stt, Vp, Vt),
    )


def clusterize(digits, n_sectors, n_rows, n_time, n_pads, thr_peak=6, noise_eps=4, cog_gated=False, cog_shared=False):
    """O0..O5.  Returns (list of cluster dicts in (sector,row,time,pad) order, bad_flag)."""
    maps, bad = build_maps(digits, n_sectors, n_rows, n_time, n_pads)
    out = []
    for (s, r) in sorted(maps):
        m = maps[(s, r)]
        T, P = n_time, n_pads[r]
        pk, rank = peaks_of(m, T, P, thr_peak)
        sv = survivors_of(m, pk, rank, noise_eps)
        for c in sorted(sv):  # (time, pad) ascending == O5 within a row
            out.append(cluster_shared_of(m, T, P, c, sv, s, r) if cog_shared else cluster_of(m, T, P, c, s, r, cog_gated))
    return out, bad


def row_flags(q, thr_peak=6, noise_eps=4):
    """bit0 peak / bit1 survivor for a small [T][P] array (mirror of t1.row_flags)."""
    q = np.asarray(q)
    T, P = q.shape
    m = {(t, p): int(q[t, p]) for t in range(T) for p in range(P) if q[t, p] > 0}
    pk, rank = peaks_of(m, T, P, thr_peak)
    sv = survivors_of(m, pk, rank, noise_eps)
    f = np.zeros((T, P), dtype=np.uint8)
    for c in pk:
        f[c] |= 1
    for c in sv:
        f[c] |= 2
    return f
