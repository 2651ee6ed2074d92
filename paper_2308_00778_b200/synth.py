"""Seeded synthetic Gaia-shaped systems (inputs only -- none of the method's arithmetic).

The paper measures on proprietary Gaia datasets that do not exist here;
BASELINE.json's configs take their *shape* (24 stored coefficients per observation row in
5/12/6/1 sections, block-diagonal astrometric part, rows grouped by star)
and this module generates such systems.  It serves both the CPU oracle's tests and the CUDA
path's tests/bench and therefore contains no aprod / LSQR arithmetic: it emits the upload
arrays (values, matrixIndexAstro, matrixIndexAtt, instrCol), x_true, the noise vector and
the constraint rows.  Forming b = A x_true + noise is left to the caller (tests use the
oracle for it, bench.py uses the library under test).

Everything is a pure function of (seed, stream, counter): a splitmix64-style finaliser over
int64 tensors, so any row range can be generated independently, on the CPU or on the GPU,
with bit-identical integer arrays.  Normal deviates use Box-Muller through torch's log/cos
and may differ by an ulp between devices: values are *inputs*; whichever device generated
them, the same bytes are handed to the library and to the oracle.
"""
from __future__ import annotations

import dataclasses
import math

import torch

N_PAR = 24
_GAMMA = -7046029254386353131          # 0x9E3779B97F4A7C15 as int64
_M1 = -4658895280553007687             # 0xBF58476D1CE4E5B9
_M2 = -7723592293110705685             # 0x94D049BB133111EB

# stream ids
S_OBSCOUNT, S_TIME, S_INSTR, S_VAL, S_XTRUE, S_NOISE, S_BURSTC, S_BURSTSEL, S_CONCOL, S_CONVAL = range(10)


def _lsr(z: torch.Tensor, k: int) -> torch.Tensor:
    return (z >> k) & ((1 << (64 - k)) - 1)


def _mix(z: torch.Tensor) -> torch.Tensor:
    z = (z ^ _lsr(z, 30)) * _M1
    z = (z ^ _lsr(z, 27)) * _M2
    return z ^ _lsr(z, 31)


def _key(seed: int, stream: int) -> int:
    z = torch.tensor([(seed * 1000003 + stream * 7919 + 1) & 0x7FFFFFFFFFFFFFFF], dtype=torch.int64)
    return int(_mix(_mix(z + _GAMMA) + _GAMMA)[0])


def hash64(seed: int, stream: int, idx: torch.Tensor) -> torch.Tensor:
    """idx: int64 tensor of counters -> int64 tensor of 64 hashed bits."""
    return _mix(idx * _GAMMA + _key(seed, stream))


def uniform(seed: int, stream: int, idx: torch.Tensor) -> torch.Tensor:
    """U[0,1) with 53 random bits."""
    return _lsr(hash64(seed, stream, idx), 11).to(torch.float64) * (2.0 ** -53)


def normal(seed: int, stream: int, idx: torch.Tensor) -> torch.Tensor:
    """N(0,1) by Box-Muller on counters 2*idx, 2*idx+1."""
    u1 = uniform(seed, stream, idx * 2)
    u2 = uniform(seed, stream, idx * 2 + 1)
    return torch.sqrt(-2.0 * torch.log1p(-u1)) * torch.cos((2.0 * math.pi) * u2)


@dataclasses.dataclass(frozen=True)
class SynthConfig:
    name: str
    n_stars: int
    n_dof_att: int                  # N_DFA per axis
    n_instr: int
    obs_per_star: int = 0           # > 0: fixed count
    obs_powerlaw: tuple | None = None   # (alpha, kmin, kmax): pdf ~ k^-alpha on [kmin, kmax]
    att_bursts: tuple | None = None     # (n_bursts, half_width, fraction_in_bursts)
    instr_zipf: float = 0.0         # > 0: Zipf exponent over the n_instr columns
    noise_sigma: float = 1e-3       # N(0, 1e-6) read as a variance (R17)
    n_con: int = 0                  # constraint rows
    con_nnz: int = 0                # distinct astro columns per constraint row
    seed: int = 0
    n_glob: int = 1                 # global columns (1 in the paper's production layout; it also ran 5)
    # section widths (0 <= N_Astro <= 5, N_Att = 12 or no attitude part, 0 <= N_Instr <= 6);
    # a section of width 0 has no columns (the paper's 40 / 100 / 300 GB datasets solve only some sections)
    n_astro_par: int = 5
    n_att_par: int = 12
    n_instr_par: int = 6

    @property
    def n(self) -> int:
        return (self.n_astro_par * self.n_stars + (3 * self.n_dof_att if self.n_att_par else 0)
                + (self.n_instr if self.n_instr_par else 0) + self.n_glob)

    @property
    def n_par(self) -> int:         # stored coefficients per row (24 in production)
        return self.n_astro_par + self.n_att_par + self.n_instr_par + self.n_glob


def tiny(seed=0):      # BASELINE.json configs[0]
    return SynthConfig("tiny", 2_000, 1_000, 2_000, obs_per_star=50, seed=seed)


def small(seed=0):     # configs[1]
    return SynthConfig("small", 200_000, 100_000, 6_000, obs_per_star=100, seed=seed)


def medium(seed=0):    # configs[2]
    return SynthConfig("medium", 1_000_000, 1_000_000, 60_000, obs_per_star=200, seed=seed)


def skewed(seed=0, alpha=2.0):    # configs[3]
    return SynthConfig("skewed", 1_000_000, 1_000_000, 60_000, obs_powerlaw=(alpha, 10, 2000),
                       att_bursts=(1000, 1e-4, 0.9), instr_zipf=1.1, seed=seed)


def large(seed=0):     # configs[4]
    return SynthConfig("large", 2_500_000, 1_000_000, 60_000, obs_per_star=200, n_con=10_000,
                       con_nnz=1_000, seed=seed)


def mini(seed=0, n_stars=20, obs=12, n_dof_att=10, n_instr=8, n_con=0, con_nnz=0):
    """Brute-force size: dense expansion fits in a few hundred KB."""
    return SynthConfig("mini", n_stars, n_dof_att, n_instr, obs_per_star=obs, n_con=n_con,
                       con_nnz=con_nnz, seed=seed)


def star_rowptr(cfg: SynthConfig, device="cpu") -> torch.Tensor:
    """int64 [n_stars+1]: first row of each star (rows are sorted by star)."""
    if cfg.obs_per_star > 0:
        return torch.arange(cfg.n_stars + 1, dtype=torch.int64, device=device) * cfg.obs_per_star
    alpha, kmin, kmax = cfg.obs_powerlaw
    u = uniform(cfg.seed, S_OBSCOUNT, torch.arange(cfg.n_stars, dtype=torch.int64, device=device))
    e = 1.0 - alpha
    a, b = float(kmin) ** e, float(kmax + 1) ** e
    k = torch.floor((a + u * (b - a)) ** (1.0 / e)).to(torch.int64).clamp_(kmin, kmax)
    rp = torch.zeros(cfg.n_stars + 1, dtype=torch.int64, device=device)
    rp[1:] = torch.cumsum(k, 0)
    return rp


def _zipf_cdf(n: int, s: float, device) -> torch.Tensor:
    w = torch.arange(1, n + 1, dtype=torch.float64, device=device) ** (-s)
    c = torch.cumsum(w, 0)
    return c / c[-1]


def _distinct_draws(seed, stream, base_idx, n_choices, width, cdf=None):
    """[r, width] int64 of distinct values per row in [0, n_choices); duplicates are redrawn
    with an incremented attempt counter (deterministic)."""
    assert n_choices >= width
    r = base_idx.shape[0]
    dev = base_idx.device
    slot = base_idx[:, None] * width + torch.arange(width, dtype=torch.int64, device=dev)[None, :]
    attempt = torch.zeros((r, width), dtype=torch.int64, device=dev)

    def draw(sl, at):
        u = uniform(seed, stream, sl * 4096 + at)
        if cdf is None:
            return torch.floor(u * n_choices).to(torch.int64).clamp_(max=n_choices - 1)
        return torch.searchsorted(cdf, u).clamp_(max=n_choices - 1)

    col = draw(slot, attempt)
    for _ in range(4095):
        dup = torch.zeros((r, width), dtype=torch.bool, device=dev)
        for j in range(1, width):
            dup[:, j] = (col[:, :j] == col[:, j:j + 1]).any(dim=1)
        if not bool(dup.any()):
            return col
        attempt = attempt + dup.to(torch.int64)
        col = torch.where(dup, draw(slot, attempt), col)
    raise RuntimeError("could not draw distinct columns")


def generate_rows(cfg: SynthConfig, star0: int, star1: int, device="cpu", rowptr=None) -> dict:
    """Upload arrays for the rows of stars [star0, star1).

    Returns dict(row0, values [r,n_par] f64, matrixIndexAstro [r] i64 (= n_astro_par*star), matrixIndexAtt [r] i64,
    instrCol [r,n_instr_par] i32, noise [r] f64).  Rows are sorted by star and by time within a star.
    """
    if rowptr is None:
        rowptr = star_rowptr(cfg, device)
    row0, row1 = int(rowptr[star0]), int(rowptr[star1])
    r = row1 - row0
    rows = torch.arange(row0, row1, dtype=torch.int64, device=device)
    counts = (rowptr[star0 + 1:star1 + 1] - rowptr[star0:star1]).to(device)
    star = torch.repeat_interleave(torch.arange(star0, star1, dtype=torch.int64, device=device), counts,
                                   output_size=r)
    # observation times
    t = uniform(cfg.seed, S_TIME, rows)
    if cfg.att_bursts is not None:
        nb, hw, frac = cfg.att_bursts
        sel = uniform(cfg.seed, S_BURSTSEL, rows * 2)
        which = torch.floor(uniform(cfg.seed, S_BURSTSEL, rows * 2 + 1) * nb).to(torch.int64).clamp_(max=nb - 1)
        centre = uniform(cfg.seed, S_BURSTC, which)
        tb = (centre + (2.0 * t - 1.0) * hw).clamp_(0.0, 1.0 - 2.0 ** -53)
        t = torch.where(sel < frac, tb, t)
    if cfg.obs_per_star > 0:
        t = torch.sort(t.view(star1 - star0, cfg.obs_per_star), dim=1).values.reshape(-1)
    else:
        t = torch.sort(star.to(torch.float64) + t).values - star.to(torch.float64)
        t = t.clamp_(0.0, 1.0 - 2.0 ** -53)
    iatt = torch.floor(t * (cfg.n_dof_att - 3)).to(torch.int64).clamp_(0, cfg.n_dof_att - 4)
    cdf = _zipf_cdf(cfg.n_instr, cfg.instr_zipf, device) if cfg.instr_zipf > 0 else None
    if cfg.n_instr_par > 0:
        ic = _distinct_draws(cfg.seed, S_INSTR, rows, cfg.n_instr, cfg.n_instr_par, cdf).to(torch.int32)
    else:
        ic = torch.zeros((r, 0), dtype=torch.int32, device=device)
    k = torch.arange(cfg.n_par, dtype=torch.int64, device=device)
    values = normal(cfg.seed, S_VAL, rows[:, None] * cfg.n_par + k[None, :])
    noise = normal(cfg.seed, S_NOISE, rows) * cfg.noise_sigma
    return dict(row0=row0, values=values, matrixIndexAstro=star * cfg.n_astro_par, matrixIndexAtt=iatt,
                instrCol=ic, noise=noise)


def x_true(cfg: SynthConfig, device="cpu") -> torch.Tensor:
    return normal(cfg.seed, S_XTRUE, torch.arange(cfg.n, dtype=torch.int64, device=device))


def constraints(cfg: SynthConfig, device="cpu"):
    """CSR (rowptr i64 [n_con+1], col i64 [nnz] absolute astro columns, val f64 [nnz])."""
    if cfg.n_con == 0:
        return (torch.zeros(1, dtype=torch.int64, device=device),
                torch.zeros(0, dtype=torch.int64, device=device),
                torch.zeros(0, dtype=torch.float64, device=device))
    rows = torch.arange(cfg.n_con, dtype=torch.int64, device=device)
    col = _distinct_draws(cfg.seed, S_CONCOL, rows, max(cfg.n_astro_par, 1) * cfg.n_stars, cfg.con_nnz)
    col = torch.sort(col, dim=1).values.reshape(-1)
    val = normal(cfg.seed, S_CONVAL, torch.arange(cfg.n_con * cfg.con_nnz, dtype=torch.int64, device=device))
    rowptr = torch.arange(cfg.n_con + 1, dtype=torch.int64, device=device) * cfg.con_nnz
    return rowptr, col, val


def generate(cfg: SynthConfig, device="cpu", chunk_stars: int = 0) -> dict:
    """Whole system at once (Tiny/Small sizes): concatenation of generate_rows chunks."""
    rp = star_rowptr(cfg, device)
    step = chunk_stars or max(1, min(cfg.n_stars, 20_000))
    parts = [generate_rows(cfg, s, min(s + step, cfg.n_stars), device, rp)
             for s in range(0, cfg.n_stars, step)]
    out = {k: torch.cat([p[k] for p in parts]) for k in
           ("values", "matrixIndexAstro", "matrixIndexAtt", "instrCol", "noise")}
    out["rowptr"] = rp
    out["x_true"] = x_true(cfg, device)
    out["con_rowptr"], out["con_col"], out["con_val"] = constraints(cfg, device)
    return out
