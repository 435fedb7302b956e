"""Seeded synthetic line lists shaped like the paper's workloads (BASELINE.json
`configs`).  INPUT DATA ONLY: this module holds none of the
method's arithmetic and is the one thing the oracle side and the CUDA side share.

The real line lists (ExoMol BT2 water, Kurucz/NIST/VALD3 atoms; PAPER.md L710,
L7, L662) are not in this container and are not reconstructed; only shapes,
sizes and value distributions are used.

Counter-based generator: u(seed, cfg, field, i) = (splitmix64(key) >> 11) * 2^-53
with key = seed*K0 + cfg*K1 + field*K2 + i (wrapping int64 arithmetic), written
with torch integer ops so the same code runs on the CPU (tests) and on the GPU
(bench, 5e8 lines).  libm differs between devices in the last ulp, so arrays are
generated ONCE, on one device, and then handed to both sides.
"""
import math

import torch

FIELDS = ("nu0", "A", "g_up", "E_low", "gamma_ref", "n_exp")
ATM_PER_BAR = 1.0 / 1.01325

_M64 = (1 << 64) - 1


def _s64(v: int) -> int:
    """python int -> value as signed 64-bit (two's complement)."""
    v &= _M64
    return v - (1 << 64) if v >= (1 << 63) else v


def _lsr(x: torch.Tensor, s: int) -> torch.Tensor:
    """logical shift right on int64 tensors."""
    return (x >> s) & ((1 << (64 - s)) - 1)


def _splitmix64(x: torch.Tensor) -> torch.Tensor:
    x = x + _s64(0x9E3779B97F4A7C15)
    x = (x ^ _lsr(x, 30)) * _s64(0xBF58476D1CE4E5B9)
    x = (x ^ _lsr(x, 27)) * _s64(0x94D049BB133111EB)
    return x ^ _lsr(x, 31)


def uniform(seed: int, cfg: int, field: int, n: int, device="cpu", start: int = 0) -> torch.Tensor:
    """n uniforms in [0,1), fp64, counters start..start+n-1."""
    base = _s64(seed * 0xD1342543DE82EF95 + cfg * 0xA0761D6478BD642F + field * 0xE7037ED1A0B428DB)
    i = torch.arange(start, start + n, dtype=torch.int64, device=device)
    bits = _splitmix64(i + base)
    return _lsr(bits, 11).to(torch.float64) * (2.0 ** -53)


def _loguniform(u, lo, hi):
    return torch.pow(10.0, math.log10(lo) + u * (math.log10(hi) - math.log10(lo)))


def _integer(u, k):
    return 1.0 + torch.floor(u * k)


def _exponential(u, mean, clip):
    return torch.clamp(-mean * torch.log1p(-u), max=clip)


CONFIGS = {
    # idx: name, n, grid (numin, numax, dnu), cut, T, P_atm, mass, Q
    1: dict(name="tiny_molecule", n=10_000, grid=(0.0, 2000.0, 0.1), cut=25.0,
            T=1000.0, P_atm=1.0, mass_amu=18.0, Q=500.0),
    2: dict(name="mid_molecule", n=1_000_000, grid=(0.0, 10000.0, 0.01), cut=25.0,
            T=1500.0, P_atm=ATM_PER_BAR, mass_amu=18.0, Q=2000.0),
    3: dict(name="bt2_shaped_coarse", n=500_000_000, grid=(0.0, 30000.0, 0.1), cut=25.0,
            T=1500.0, P_atm=1.0, mass_amu=18.015, Q=3000.0),
    4: dict(name="bt2_shaped_fine", n=500_000_000, grid=(0.0, 30000.0, 0.01), cut=100.0,
            T=2000.0, P_atm=10.0 * ATM_PER_BAR, mass_amu=18.015, Q=6000.0),
    5: dict(name="atom_like_uncut", n=200_000, grid=(0.0, 50000.0, 0.01), cut=0.0,
            T=2500.0, P_atm=ATM_PER_BAR, mass_amu=55.845, Q=50.0),
}


def _centres(cfg, seed, n, device):
    gen = 3 if cfg == 4 else cfg          # configs 3 and 4 share the generator and seed
    u = uniform(seed, gen, 0, n, device)
    if cfg == 1:
        return torch.sort(u * 2000.0).values
    if cfg == 2:
        # 40 % uniform on [0, 1e4); 3 clusters x 20 %, sigma 300 (R17); unsorted
        nu = uniform(seed, gen, 7, n, device) * 10000.0
        centres = (1600.0, 3750.0, 7250.0)
        for k, c in enumerate(centres):
            sel = (u >= 0.2 * k) & (u < 0.2 * (k + 1))
            ok = torch.zeros_like(sel)
            for attempt in range(8):      # redraw samples outside the range
                u1 = uniform(seed, gen, 8 + 2 * attempt, n, device)
                u2 = uniform(seed, gen, 9 + 2 * attempt, n, device)
                z = torch.sqrt(-2.0 * torch.log1p(-u1)) * torch.cos(2.0 * math.pi * u2)
                cand = c + 300.0 * z
                take = sel & ~ok & (cand >= 0.0) & (cand < 10000.0)
                nu = torch.where(take, cand, nu)
                ok = ok | take
        return nu
    if cfg in (3, 4):
        s, R = 8000.0, 30000.0
        nu = -s * torch.log1p(-u * (1.0 - math.exp(-R / s)))
        return torch.sort(nu).values
    if cfg == 5:
        return u * 50000.0
    raise ValueError(cfg)


_FIELD_SPECS = {
    # cfg: (A lo, A hi, g max, E kind, E p1, E p2, gamma lo, gamma hi)
    1: (1e-6, 1e2, 50, "uniform", 0.0, 15000.0, 0.01, 0.1),
    2: (1e-8, 1e2, 100, "exp", 5000.0, 30000.0, 0.01, 0.1),
    3: (1e-10, 1e3, 150, "exp", 8000.0, 40000.0, 0.02, 0.1),
    5: (1e2, 1e9, 20, "uniform", 0.0, 60000.0, 0.05, 0.5),
}


def make_lines(cfg: int, n: int = None, seed: int = 0, device="cpu"):
    """The six fp64 SoA line arrays of config `cfg` (1..5), optionally with a
    reduced line count n (a 'mini twin': same generator, fewer lines)."""
    gen = 3 if cfg == 4 else cfg
    if n is None:
        n = CONFIGS[cfg]["n"]
    Alo, Ahi, gmax, Ekind, E1, E2, glo, ghi = _FIELD_SPECS[gen]
    out = {"nu0": _centres(cfg, seed, n, device)}
    out["A"] = _loguniform(uniform(seed, gen, 1, n, device), Alo, Ahi)
    out["g_up"] = _integer(uniform(seed, gen, 2, n, device), gmax)
    uE = uniform(seed, gen, 3, n, device)
    out["E_low"] = E1 + uE * (E2 - E1) if Ekind == "uniform" else _exponential(uE, E1, E2)
    out["gamma_ref"] = glo + uniform(seed, gen, 4, n, device) * (ghi - glo)
    out["n_exp"] = 0.5 + uniform(seed, gen, 5, n, device) * 0.25
    return out


def conditions(cfg: int):
    c = CONFIGS[cfg]
    return {k: c[k] for k in ("T", "P_atm", "mass_amu", "Q")}


def to_numpy(lines):
    return {k: v.detach().cpu().numpy() for k, v in lines.items()}


# ---- HITRAN-shaped list: the mid-molecule generator plus the extra HITRAN columns -------------
HITRAN_FIELDS = ("nu0", "A", "g_up", "E_low", "gamma_air", "gamma_self", "n_exp", "delta")
HITRAN_ISOS = ((18.0106, 2000.0, 0.99732), (20.0148, 2016.0, 0.00200), (19.0148, 11940.0, 0.00037))   # mass, Q, abundance
HITRAN_COND = dict(T=1500.0, P_atm=5.0, P_self_atm=0.5, isos=HITRAN_ISOS)


def make_lines_hitran(n: int, seed: int = 0, device="cpu"):
    """Config-2-shaped centres and strengths; gamma_air as gamma_ref, gamma_self 2-5 x gamma_air, pressure shift
    uniform on [-0.02, 0.01] cm^-1/atm, isotopologue 0 / 1 / 2 with probability 0.95 / 0.03 / 0.02.  Unsorted."""
    base = make_lines(2, n=n, seed=seed, device=device)
    out = {k: base[k] for k in ("nu0", "A", "g_up", "E_low", "n_exp")}
    out["gamma_air"] = base["gamma_ref"]
    out["gamma_self"] = base["gamma_ref"] * (2.0 + 3.0 * uniform(seed, 2, 40, n, device))
    out["delta"] = -0.02 + 0.03 * uniform(seed, 2, 41, n, device)
    u = uniform(seed, 2, 42, n, device)
    out["iso"] = ((u >= 0.95).to(torch.int32) + (u >= 0.98).to(torch.int32))
    return out
