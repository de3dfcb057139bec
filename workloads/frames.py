"""Seeded synthetic TPC time frames (the five BASELINE.json configs).

This module is the ONLY code shared by the oracle side and the CUDA side of
the tests and the bench: it makes inputs and holds none of the clusterizer's
arithmetic (no map, no peak test, no centre of gravity).  Plain torch ops, so
the same recipe runs on the CPU (small configs, CPU tests) and on the GPU
(full time frames: 8e9 cells are generated sector by sector in HBM).

The frames stand in for the paper's workload, "a reference MC time frame with
100 Pb-Pb collisions" and real 2022-24 data, neither of
which exists here.  Recipe: SURVEY.md 8(d) / DESIGN.md "Input recipe".

Digit record, packed little-endian into one int64:
  charge | time << 16 | pad << 32 | row << 40 | sector << 48
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np
import torch

SEED_BASE = 251117018  # seed_k = SEED_BASE + k
ZS_THRESHOLD = 3       # zero suppression: cells < 3 ADC are dropped


def n_pads_ramp(n_rows: int = 152) -> np.ndarray:
    """Q1: pads per row ramping linearly 66 -> 138 (sum 15504 for 152 rows)."""
    r = np.arange(n_rows, dtype=np.int64)
    return (66 + (72 * r + 75) // 151).astype(np.uint16)


# Cluster densities (injected clusters per map cell) were calibrated by
# bisection on a reduced geometry (recipe in
# DESIGN.md "Input recipe") so that occupancy after zero suppression hits the target within
# +-2 % relative, then frozen here.
CONFIGS = {
    0: dict(name="cfg0-single-sector", n_sectors=1, n_rows=152, n_time=512, pads="const96",
            n_clusters=2000, sigma_p=(0.8, 0.8), sigma_t=(1.0, 1.0), amp="exp40", noise=1.0),
    1: dict(name="cfg1-adversarial", n_sectors=1, n_rows=16, n_time=256, pads="const64",
            n_clusters=400, sigma_p=(0.8, 0.8), sigma_t=(1.0, 1.0), amp="exp40", noise=1.0),
    2: dict(name="cfg2-full-geometry-short", n_sectors=36, n_rows=152, n_time=2000, pads="ramp",
            density=8.36e-3, sigma_p=(0.8, 0.8), sigma_t=(1.0, 1.0), amp="exp40", noise=1.0,
            target_occupancy=0.10),
    3: dict(name="cfg3-pp-like", n_sectors=36, n_rows=152, n_time=14256, pads="ramp",
            density=3.266e-4, sigma_p=(0.8, 0.8), sigma_t=(1.0, 1.0), amp="exp40", noise=1.0,
            target_occupancy=0.01),
    4: dict(name="cfg4-pbpb-like", n_sectors=36, n_rows=152, n_time=14256, pads="ramp",
            density=8.47e-3, sigma_p=(0.6, 1.4), sigma_t=(0.8, 1.6), amp="moyal", noise=1.2,
            target_occupancy=0.20),
}


@dataclass
class Frame:
    digits: torch.Tensor          # int64 [n], packed 8-byte records
    n_sectors: int
    n_rows: int
    n_time: int
    n_pads: np.ndarray            # uint16 [n_rows]
    meta: dict = field(default_factory=dict)

    @property
    def n_digits(self) -> int:
        return int(self.digits.numel())

    @property
    def cells(self) -> int:
        return int(self.n_sectors) * int(self.n_time) * int(self.n_pads.astype(np.int64).sum())

    def digits_numpy(self) -> np.ndarray:
        """uint64 host copy; ``.view`` it with the 8-byte record dtype of either side."""
        return self.digits.cpu().numpy().view(np.uint64)


def pack_digits(sector, row, pad, time, charge) -> torch.Tensor:
    return (charge.to(torch.int64) | (time.to(torch.int64) << 16) | (pad.to(torch.int64) << 32)
            | (row.to(torch.int64) << 40) | (sector.to(torch.int64) << 48))


def checksum(digits: torch.Tensor) -> int:
    """64-bit order-independent checksum: wrapping sum of a mix of every record."""
    x = digits
    x = (x ^ (x >> 31)) * 0x7FB5D329728EA185
    x = (x ^ (x >> 27)) * (-0x7E25210B43D22BB3)
    x = x ^ (x >> 33)
    return int(x.sum().item()) & 0xFFFFFFFFFFFFFFFF


def _pads_of(cfg) -> np.ndarray:
    if cfg["pads"] == "ramp":
        return n_pads_ramp(cfg["n_rows"])
    return np.full(cfg["n_rows"], int(cfg["pads"][5:]), dtype=np.uint16)


def _amplitudes(kind: str, n: int, g: torch.Generator, device) -> torch.Tensor:
    if kind == "exp40":   # A ~ Exp(mean 40)
        u = torch.rand(n, generator=g, device=device, dtype=torch.float64)
        return (-40.0 * torch.log1p(-u)).float()
    if kind == "moyal":   # Landau-like: A = 44.76 + 12 * (-ln z^2), z ~ N(0,1), clipped [1,4000]
        z = torch.randn(n, generator=g, device=device, dtype=torch.float64)
        a = 44.76 + 12.0 * (-torch.log(z * z + 1e-300))
        return a.clamp_(1.0, 4000.0).float()
    raise ValueError(kind)


def _inject(signal: torch.Tensor, row_off: torch.Tensor, pads_t: torch.Tensor, T: int,
            row, p0, t0, amp, sp, st, chunk: int = 1 << 17) -> None:
    """Add Gaussian clusters (fixed point, 1/256 ADC, integer adds -> order-free).

    signal: int32 [sector_cells] in [row][time][pad] order; the value added at
    a cell centre (p,t) is A*exp(-((p-p0)^2/sp^2 + (t-t0)^2/st^2)/2) within +-4 sigma.
    """
    dev = signal.device
    wp = int(math.ceil(4.0 * float(sp.max()))) + 1 if sp.numel() else 1
    wt = int(math.ceil(4.0 * float(st.max()))) + 1 if st.numel() else 1
    dp = torch.arange(-wp, wp + 1, device=dev)
    dt = torch.arange(-wt, wt + 1, device=dev)
    for a in range(0, row.numel(), chunk):
        b = min(a + chunk, row.numel())
        r = row[a:b]
        P = pads_t[r]                                             # [c]
        pc = torch.floor(p0[a:b]).long()[:, None] + dp[None, :]   # [c, np]
        tc = torch.floor(t0[a:b]).long()[:, None] + dt[None, :]   # [c, nt]
        xp = (pc.float() - p0[a:b, None]) / sp[a:b, None]
        xt = (tc.float() - t0[a:b, None]) / st[a:b, None]
        okp = (xp.abs() <= 4.0) & (pc >= 0) & (pc < P[:, None])
        okt = (xt.abs() <= 4.0) & (tc >= 0) & (tc < T)
        gp = torch.exp(-0.5 * xp * xp)
        gt = torch.exp(-0.5 * xt * xt)
        val = amp[a:b, None, None] * gt[:, :, None] * gp[:, None, :]          # [c, nt, np]
        ok = okt[:, :, None] & okp[:, None, :]
        idx = row_off[r][:, None, None] + tc[:, :, None] * P[:, None, None] + pc[:, None, :]
        v = torch.round(val * 256.0).to(torch.int32)
        ok &= v != 0
        signal.index_add_(0, idx[ok], v[ok])


def _digitize(signal: torch.Tensor, noise_sigma: float, g: torch.Generator, stamp=None):
    """signal/256 + N(0,sigma) -> round -> clip [0,1023] -> zero suppression.

    Returns (flat cell index int64 [n], charge int64 [n]) in ascending cell order.
    """
    v = signal.float() / 256.0
    v += torch.randn(v.shape, generator=g, device=v.device, dtype=torch.float32) * noise_sigma
    v = torch.round(v).clamp_(0, 1023).to(torch.int16)
    if stamp is not None:  # CFG[1]: equal-charge blocks stamped AFTER noise so ties survive
        idx, val = stamp
        v.scatter_reduce_(0, idx, val.to(torch.int16), "amax", include_self=True)
    keep = v >= ZS_THRESHOLD
    cell = keep.nonzero(as_tuple=False).squeeze(1)
    return cell, v[cell].to(torch.int64)


def _cells_to_fields(cell, row_off, pads_t, T):
    row = torch.searchsorted(row_off, cell, right=True) - 1
    rem = cell - row_off[row]
    P = pads_t[row]
    time = rem // P
    pad = rem - time * P
    return row, pad, time


def _row_tables(pads: np.ndarray, T: int, device):
    pads_t = torch.as_tensor(pads.astype(np.int64), device=device)
    row_off = torch.zeros(len(pads) + 1, dtype=torch.int64, device=device)
    row_off[1:] = torch.cumsum(pads_t * T, 0)
    return pads_t, row_off


def _sector_generator(seed: int, sector: int, device) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed((seed * 1000003 + sector * 7919 + 12345) & 0x7FFFFFFFFFFFFFFF)
    return g


def _gen_sector_standard(cfg, pads, sector, n_clusters, seed, device, rows_subset=None):
    """One sector of CFG[0,2,3,4]: uniform clusters + noise. Returns packed digits (cell order)."""
    T = cfg["n_time"]
    pads_t, row_off = _row_tables(pads, T, device)
    g = _sector_generator(seed, sector, device)
    w = pads_t.double()
    row = torch.multinomial(w / w.sum(), n_clusters, replacement=True, generator=g) if n_clusters else \
        torch.zeros(0, dtype=torch.int64, device=device)
    u = torch.rand((4, n_clusters), generator=g, device=device)
    p0 = u[0] * pads_t[row].float()
    t0 = u[1] * float(T)
    sp = cfg["sigma_p"][0] + (cfg["sigma_p"][1] - cfg["sigma_p"][0]) * u[2]
    st = cfg["sigma_t"][0] + (cfg["sigma_t"][1] - cfg["sigma_t"][0]) * u[3]
    amp = _amplitudes(cfg["amp"], n_clusters, g, device)
    signal = torch.zeros(int(row_off[-1]), dtype=torch.int32, device=device)
    _inject(signal, row_off, pads_t, T, row, p0, t0, amp, sp, st)
    cell, q = _digitize(signal, cfg["noise"], g)
    del signal
    r, p, t = _cells_to_fields(cell, row_off, pads_t, T)
    truth = dict(row=row, p0=p0, t0=t0, amp=amp, sp=sp, st=st)
    return pack_digits(torch.full_like(r, sector), r, p, t, q), truth


def _gen_cfg1(cfg, pads, seed, device):
    """Tie/edge adversarial map (SURVEY 8(d) table, row cfg 1)."""
    T, R = cfg["n_time"], cfg["n_rows"]
    pads_t, row_off = _row_tables(pads, T, device)
    g = _sector_generator(seed, 0, device)
    n_seed, n_fol = 100, 3
    P = int(pads[0])
    srow = torch.randint(0, R, (n_seed,), generator=g, device=device)
    sp0 = torch.rand(n_seed, generator=g, device=device) * P
    st0 = torch.rand(n_seed, generator=g, device=device) * T
    # 10 % of the seed centres forced onto a pad or time edge
    edge = torch.rand(n_seed, generator=g, device=device) < 0.10
    which = torch.randint(0, 8, (n_seed,), generator=g, device=device)
    pe = torch.tensor([0.0, 1.0, P - 2.0, P - 1.0], device=device)
    te = torch.tensor([0.0, 1.0, T - 2.0, T - 1.0], device=device)
    sp0 = torch.where(edge & (which < 4), pe[which % 4], sp0)
    st0 = torch.where(edge & (which >= 4), te[which % 4], st0)
    ang = torch.rand((n_seed, n_fol), generator=g, device=device) * (2 * math.pi)
    dist = 1.0 + 2.0 * torch.rand((n_seed, n_fol), generator=g, device=device)   # 1..3 bins
    row = torch.cat([srow, srow.repeat_interleave(n_fol)])
    p0 = torch.cat([sp0, (sp0[:, None] + dist * torch.cos(ang)).reshape(-1)]).clamp_(0, P - 1e-3)
    t0 = torch.cat([st0, (st0[:, None] + dist * torch.sin(ang)).reshape(-1)]).clamp_(0, T - 1e-3)
    n = row.numel()  # 400
    amp = _amplitudes(cfg["amp"], n, g, device)
    kind = torch.rand(n, generator=g, device=device)
    plateau = kind < 0.20
    saturated = (kind >= 0.20) & (kind < 0.25)
    amp = torch.where(saturated, torch.full_like(amp, 3000.0), amp)
    gauss = ~plateau
    sp = torch.full((n,), cfg["sigma_p"][0], device=device)
    st = torch.full((n,), cfg["sigma_t"][0], device=device)
    signal = torch.zeros(int(row_off[-1]), dtype=torch.int32, device=device)
    _inject(signal, row_off, pads_t, T, row[gauss], p0[gauss], t0[gauss], amp[gauss], sp[gauss], st[gauss])
    # plateaus: equal-charge 2x1 (pad), 1x2 (time), 2x2 blocks, integer charge 20..200
    pr = row[plateau]
    pp = torch.floor(p0[plateau]).long().clamp_(0, P - 2)
    pt = torch.floor(t0[plateau]).long().clamp_(0, T - 2)
    shape = torch.randint(0, 3, (pr.numel(),), generator=g, device=device)
    val = torch.randint(20, 201, (pr.numel(),), generator=g, device=device)
    idx, vals = [], []
    for (dp_, dt_, sel) in ((0, 0, None), (1, 0, (0, 2)), (0, 1, (1, 2)), (1, 1, (2,))):
        m = torch.ones_like(shape, dtype=torch.bool) if sel is None else \
            torch.stack([shape == s_ for s_ in sel]).any(0)
        idx.append((row_off[pr] + (pt + dt_) * P + (pp + dp_))[m])
        vals.append(val[m])
    cell, q = _digitize(signal, cfg["noise"], g, stamp=(torch.cat(idx), torch.cat(vals)))
    r, p, t = _cells_to_fields(cell, row_off, pads_t, T)
    truth = dict(row=row, p0=p0, t0=t0, amp=amp, plateau=plateau, saturated=saturated)
    return pack_digits(torch.zeros_like(r), r, p, t, q), truth


def _feistel_perm(n: int, seed: int, device) -> torch.Tensor:
    """A seeded bijection of [0, n) from elementwise ops only: a 6-round Feistel network on
    the next even power-of-two domain, cycle-walked back into range.  Used for the full
    time frames, where torch.randperm (n >= 2^30 on CUDA) takes many minutes."""
    k = max(2, (n - 1).bit_length())
    k += k & 1
    h = k // 2
    mask = (1 << h) - 1
    keys = [((seed + 0x9E3779B1 * (r + 1)) * 0x85EBCA6B) & 0x7FFFFFFF for r in range(6)]

    def f(x):
        L, R = x >> h, x & mask
        for key in keys:
            y = (R * 0x2545F491 + key) & 0xFFFFFFFFFFFF          # < 2^48: no int64 overflow
            y = ((y ^ (y >> 15)) * 0x2C1B3C6D) & 0xFFFFFFFFFFFF
            y = (y ^ (y >> 13)) & mask
            L, R = R, L ^ y
        return (L << h) | R

    x = f(torch.arange(n, dtype=torch.int64, device=device))
    bad = (x >= n).nonzero(as_tuple=False).squeeze(1)
    while bad.numel():
        v = f(x[bad])
        x[bad] = v
        bad = bad[v >= n]
    return x


def _order(digits: torch.Tensor, order: str, seed: int) -> torch.Tensor:
    """Q23 input order.  'shuffled': one global seeded permutation (headline).
    'readout': grouped by sector, then 128-bin time slab, shuffled inside."""
    n = digits.numel()
    if n == 0 or order == "cell":
        return digits
    if n >= (1 << 28):
        perm = _feistel_perm(n, seed, digits.device)
    else:
        g = torch.Generator(device=digits.device)
        g.manual_seed((seed * 2654435761 + 97) & 0x7FFFFFFFFFFFFFFF)
        perm = torch.randperm(n, generator=g, device=digits.device)
    if order == "shuffled":
        return digits[perm]
    if order == "readout":
        d = digits[perm]
        key = ((d >> 48) & 0xFF) * 1024 + (((d >> 16) & 0xFFFF) >> 7)
        return d[torch.argsort(key, stable=True)]
    raise ValueError(order)


def make_frame(k: int, device="cpu", order: str = "shuffled", seed: int | None = None,
               sectors=None, n_time: int | None = None, keep_truth: bool = False) -> Frame:
    """Build config k.  ``sectors``/``n_time`` cut a full-geometry config down
    (same per-cell density) for CPU tests and bounded CPU baselines."""
    cfg = dict(CONFIGS[k])
    seed = SEED_BASE + k if seed is None else seed
    if n_time is not None:
        cfg["n_time"] = n_time
    pads = _pads_of(cfg)
    device = torch.device(device)
    truth = None
    if k == 1:
        digits, truth = _gen_cfg1(cfg, pads, seed, device)
        n_inj = 400
    else:
        sec = list(range(cfg["n_sectors"])) if sectors is None else list(sectors)
        cells_per_sector = int(pads.astype(np.int64).sum()) * cfg["n_time"]
        n_per = cfg["n_clusters"] if "n_clusters" in cfg else int(round(cfg["density"] * cells_per_sector))
        parts = []
        for s in sec:
            d, truth = _gen_sector_standard(cfg, pads, s, n_per, seed, device)
            parts.append(d)
        digits = torch.cat(parts) if len(parts) > 1 else parts[0]
        del parts
        n_inj = n_per * len(sec)
    digits = _order(digits, order, seed)
    fr = Frame(digits=digits, n_sectors=cfg["n_sectors"], n_rows=cfg["n_rows"], n_time=cfg["n_time"],
               n_pads=pads)
    n_sec_gen = 1 if k == 1 else len(sec)
    gen_cells = n_sec_gen * cfg["n_time"] * int(pads.astype(np.int64).sum())
    fr.meta = dict(config=k, name=cfg["name"], seed=seed, order=order, injected_clusters=n_inj,
                   sectors_generated=n_sec_gen, occupancy=fr.n_digits / max(gen_cells, 1),
                   checksum=checksum(digits) if fr.n_digits else 0)
    if keep_truth:
        fr.meta["truth"] = truth
    return fr
