"""synth -- seeded synthetic matching-LP inputs shaped like the paper's workloads.

The one module both the oracle side and the CUDA side consume.  It holds NONE of the method's
arithmetic (no projection, no gradient, no step rule): only the input recipe of BASELINE.json's five
configs (restated in DESIGN.md "Input recipe"), their "tight" companions (right-hand side by the
paper's greedy-load rule, App. A) and seeded probe points.

Random numbers come from a counter-based generator (a splitmix64-style hash of (seed, stream, user,
slot)) written with torch int64 ops, so the integer streams -- degrees, item choices, and every
uniform variate -- are bit-identical on CPU and CUDA and independent of chunking.  LogNormal / Normal
variates go through log/cos and may differ in the last ulp between devices; both sides always
consume the SAME generated arrays (the oracle gets a device->host copy), never a regeneration.

Arrays produced (the ABI layout): row_ptr int64[I+1], item_idx int32[nnz] (ascending within a row),
c fp32[nnz], a fp32[nnz*m] (a[p*m+k]), b fp32[J*m] (b[j*m+k]).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace

import numpy as np
import torch

# stream ids of the counter-based generator
_S_DEG, _S_ITEM, _S_C, _S_A, _S_PERM, _S_RHO, _S_LAM, _S_NOISE, _S_NOISE2, _S_C2 = range(1, 11)

_M1 = -0x40A7B892E31B1A47  # 0xBF58476D1CE4E5B9 as int64
_M2 = -0x6B2FB644ECCEEE15  # 0x94D049BB133111EB as int64
_GOLD = -0x61C8864680B583EB  # 0x9E3779B97F4A7C15 as int64


def _lsr(x: torch.Tensor, s: int) -> torch.Tensor:
    """logical shift right on int64."""
    return (x >> s) & ((1 << (64 - s)) - 1)


def _mix(x: torch.Tensor) -> torch.Tensor:
    x = (x ^ _lsr(x, 30)) * _M1
    x = (x ^ _lsr(x, 27)) * _M2
    return x ^ _lsr(x, 31)


def _hash(seed: int, stream: int, a: torch.Tensor, b=None) -> torch.Tensor:
    """64 well-mixed bits per element keyed by (seed, stream, a[, b])."""
    k0 = ((seed * 0x9E3779B97F4A7C15 + stream * 0xD1B54A32D192ED03 + 0x2545F4914F6CDD1D) % (1 << 64))
    if k0 >= 1 << 63:
        k0 -= 1 << 64
    h = _mix(a + k0)
    if b is not None:
        h = _mix(h + b * _GOLD + 1)
    return _mix(h + _GOLD)


def _uniform(seed: int, stream: int, a: torch.Tensor, b=None) -> torch.Tensor:
    """U[0,1) in fp64 with 53 random bits; exact on every device."""
    return _lsr(_hash(seed, stream, a, b), 11).to(torch.float64) * (1.0 / (1 << 53))


def _normal(seed: int, s1: int, s2: int, a: torch.Tensor, b=None) -> torch.Tensor:
    u1 = 1.0 - _uniform(seed, s1, a, b)  # (0,1]
    u2 = _uniform(seed, s2, a, b)
    return torch.sqrt(-2.0 * torch.log(u1)) * torch.cos(2.0 * math.pi * u2)


@dataclass(frozen=True)
class Config:
    """One workload recipe (BASELINE.json configs)."""
    name: str
    I: int
    J: int
    m: int = 1
    deg: tuple = ("const", 10)          # ("const",d) | ("uniform",lo,hi) | ("poisson",mean,lo,hi)
    item: tuple = ("uniform",)          # ("uniform",) | ("zipf", s)
    c_dist: str = "uniform"             # c = -U(0,1) | c = -LogNormal(0,1)
    a_dist: str = "uniform"             # a ~ U(0.5,1.5) | a = -c | m=2: (U(0.5,1.5), 1)
    kappa: tuple = (0.2,)               # b[j,k] = kappa_k * sum_i a^k_ij
    rhs: str = "kappa"                  # "kappa" (BASELINE.json verbatim) | "greedy" (App. A)
    proj: str = "simplex"               # "simplex" | "boxcut" | "box"
    proj_params: tuple = (1.0,)         # simplex: (z,) ; boxcut: (ub, z) ; box: (lo, hi)
    gammas: tuple = (1e-2,)
    iters: tuple = (200,)
    seed: int = 0


CONFIGS = {
    "cfg1": Config("cfg1", I=1_000, J=50, deg=("const", 10), kappa=(0.2,), gammas=(1e-2,), iters=(200,)),
    "cfg2": Config("cfg2", I=1_000_000, J=1_000, deg=("uniform", 5, 35), kappa=(0.3,), gammas=(1e-3,), iters=(500,)),
    "cfg3": Config("cfg3", I=10_000_000, J=10_000, deg=("poisson", 50, 1, 400), item=("zipf", 1.1),
                   c_dist="lognormal", a_dist="neg_c", kappa=(0.25,), proj="boxcut", proj_params=(1.0, 1.0),
                   gammas=(1e-3,), iters=(1000,)),
    "cfg4": Config("cfg4", I=50_000_000, J=5_000, m=2, deg=("uniform", 50, 150), a_dist="budget_freq",
                   kappa=(0.3, 0.2), gammas=(1e-3,), iters=(300,)),
    "cfg5": Config("cfg5", I=20_000_000, J=20_000, deg=("poisson", 30, 1, 200), item=("zipf", 1.0),
                   kappa=(0.3,), proj="boxcut", proj_params=(1.0, 1.0),
                   gammas=(1e-1, 1e-2, 1e-3, 1e-4), iters=(200, 200, 200, 200)),
}


# Not a BASELINE.json config: a stress recipe for rows far beyond the streaming kernel's stage capacity (the paper's own fused
# kernel stops at 8192 nonzeros per column) -- 8,000 users with exactly 20,000 eligible items each out of 40,000.
CONFIGS["long20k"] = Config("long20k", I=8_000, J=40_000, deg=("const", 20_000), kappa=(0.3,), gammas=(1e-3,), iters=(100,))


def get_config(name: str, I: int | None = None, **over) -> Config:
    """`cfgN`, `cfgN-tight`; I=... scales the number of users (items, degrees, values keep their recipe)."""
    tight = name.endswith("-tight")
    cfg = CONFIGS[name[:-6] if tight else name]
    if tight:
        cfg = replace(cfg, name=name, rhs="greedy")
    if I is not None:
        cfg = replace(cfg, I=int(I))
    return replace(cfg, **over) if over else cfg


@dataclass
class Instance:
    cfg: Config
    row_ptr: torch.Tensor
    item_idx: torch.Tensor
    c: torch.Tensor
    a: torch.Tensor
    b: torch.Tensor
    short_rows: int = 0                 # rows whose realised degree fell below the drawn one
    meta: dict = field(default_factory=dict)

    @property
    def I(self): return self.cfg.I
    @property
    def J(self): return self.cfg.J
    @property
    def m(self): return self.cfg.m
    @property
    def nnz(self): return int(self.item_idx.numel())

    def numpy(self) -> dict:
        return {k: getattr(self, k).detach().cpu().numpy() for k in ("row_ptr", "item_idx", "c", "a", "b")}


def _degrees(cfg: Config, users: torch.Tensor) -> torch.Tensor:
    kind = cfg.deg[0]
    if kind == "const":
        return torch.full_like(users, int(cfg.deg[1]))
    u = _uniform(cfg.seed, _S_DEG, users)
    if kind == "uniform":
        lo, hi = int(cfg.deg[1]), int(cfg.deg[2])
        return lo + torch.clamp((u * (hi - lo + 1)).to(torch.int64), max=hi - lo)
    if kind == "poisson":  # inversion on a CDF table built once on the host in fp64; clipped, not resampled
        mean, lo, hi = float(cfg.deg[1]), int(cfg.deg[2]), int(cfg.deg[3])
        kmax = int(mean + 12.0 * math.sqrt(mean) + 20)
        k = np.arange(kmax + 1)
        logp = -mean + k * math.log(mean) - np.array([math.lgamma(t + 1.0) for t in k])
        cdf = torch.from_numpy(np.minimum(np.cumsum(np.exp(logp)), 1.0)).to(users.device)
        return torch.clamp(torch.searchsorted(cdf, u, right=True), min=lo, max=hi)
    raise ValueError(kind)


def _item_tables(cfg: Config, device):
    """(cdf over ranks or None, rank->item permutation or None)."""
    if cfg.item[0] == "uniform":
        return None, None
    s = float(cfg.item[1])
    w = np.arange(1, cfg.J + 1, dtype=np.float64) ** (-s)
    cdf = np.cumsum(w) / w.sum()
    cdf[-1] = 1.0
    # seeded rank -> item id permutation, so hot items are not adjacent ids
    keys = _hash(cfg.seed, _S_PERM, torch.arange(cfg.J, dtype=torch.int64))
    perm = torch.argsort(keys, stable=True)
    return torch.from_numpy(cdf).to(device), perm.to(device)


def _rows_chunk(cfg: Config, u0: int, u1: int, device, tables):
    """Eligible items of users [u0,u1): the first deg_i DISTINCT items of an i.i.d. draw sequence
    (= sequential sampling with duplicates rejected), then sorted ascending within the row."""
    cdf, perm = tables
    users = torch.arange(u0, u1, dtype=torch.int64, device=device)
    deg = torch.clamp(_degrees(cfg, users), max=cfg.J)
    over = 1.5 if cfg.item[0] == "uniform" else 3.0
    ndraw = torch.clamp((deg.to(torch.float64) * over).ceil().to(torch.int64) + 16, max=max(4 * cfg.J, 64))
    off = torch.cumsum(ndraw, 0) - ndraw
    total = int(ndraw.sum())
    row = torch.repeat_interleave(torch.arange(u1 - u0, device=device), ndraw, output_size=total)
    slot = torch.arange(total, device=device) - off[row]
    r = _uniform(cfg.seed, _S_ITEM, users[row], slot)
    if cdf is None:
        item = torch.clamp((r * cfg.J).to(torch.int64), max=cfg.J - 1)
    else:
        item = perm[torch.clamp(torch.searchsorted(cdf, r, right=True), max=cfg.J - 1)]
    key = row * cfg.J + item
    skey, order = torch.sort(key, stable=True)                     # equal keys keep draw order
    first = torch.ones(total, dtype=torch.bool, device=device)
    first[1:] = skey[1:] != skey[:-1]
    is_first = torch.zeros(total, dtype=torch.bool, device=device)
    is_first[order[first]] = True                                  # first occurrence of (row,item) in draw order
    csum = torch.cumsum(is_first.to(torch.int64), 0)
    rank = csum - (csum[off] - is_first[off].to(torch.int64))[row]  # 1-based rank among the row's distinct draws
    keep = is_first & (rank <= deg[row])
    kkey = torch.sort(key[keep]).values                            # ascending item within row
    krow = kkey // cfg.J
    real_deg = torch.bincount(krow, minlength=u1 - u0)
    short = int((real_deg < deg).sum())
    return real_deg, (kkey - krow * cfg.J).to(torch.int32), users[krow], short


def _values(cfg: Config, user: torch.Tensor, item: torch.Tensor):
    """c[nnz] fp32 and a[nnz*m] fp32, keyed by (user,item) so they do not depend on chunking."""
    it = item.to(torch.int64)
    if cfg.c_dist == "uniform":
        val = _uniform(cfg.seed, _S_C, user, it)
    elif cfg.c_dist == "lognormal":
        val = torch.exp(_normal(cfg.seed, _S_C, _S_C2, user, it))
    else:
        raise ValueError(cfg.c_dist)
    c = (-val).to(torch.float32)
    if cfg.a_dist == "uniform":
        a = (0.5 + _uniform(cfg.seed, _S_A, user, it)).to(torch.float32)
    elif cfg.a_dist == "neg_c":
        a = -c
    elif cfg.a_dist == "budget_freq":
        a1 = (0.5 + _uniform(cfg.seed, _S_A, user, it)).to(torch.float32)
        a = torch.stack([a1, torch.ones_like(a1)], dim=1).reshape(-1)
    else:
        raise ValueError(cfg.a_dist)
    return c, a


def generate(cfg: Config | str, device="cpu", chunk_users: int = 500_000) -> Instance:
    """Materialise one instance on `device` (CPU for tests, CUDA for the large configs)."""
    if isinstance(cfg, str):
        cfg = get_config(cfg)
    device = torch.device(device)
    tables = _item_tables(cfg, device)
    # the drawn degrees bound the realised ones, so the outputs can be allocated once and filled chunk by chunk
    # (config 4 is 80 GB of row data: concatenating per-chunk pieces would need twice that)
    cap = 0
    for u0 in range(0, cfg.I, chunk_users):
        users = torch.arange(u0, min(cfg.I, u0 + chunk_users), dtype=torch.int64, device=device)
        cap += int(torch.clamp(_degrees(cfg, users), max=cfg.J).sum())
    item_idx = torch.empty(cap, dtype=torch.int32, device=device)
    c = torch.empty(cap, dtype=torch.float32, device=device)
    a = torch.empty(cap * cfg.m, dtype=torch.float32, device=device)
    row_ptr = torch.zeros(cfg.I + 1, dtype=torch.int64, device=device)
    short, pos = 0, 0
    for u0 in range(0, cfg.I, chunk_users):
        u1 = min(cfg.I, u0 + chunk_users)
        d, it, usr, sh = _rows_chunk(cfg, u0, u1, device, tables)
        cc, aa = _values(cfg, usr, it)
        n = int(it.numel())
        item_idx[pos:pos + n] = it; c[pos:pos + n] = cc; a[pos * cfg.m:(pos + n) * cfg.m] = aa
        row_ptr[u0 + 1:u1 + 1] = torch.cumsum(d, 0) + pos
        pos += n
        short += sh
        del d, it, usr, cc, aa
    item_idx, c, a = item_idx[:pos], c[:pos], a[:pos * cfg.m]
    inst = Instance(cfg, row_ptr, item_idx, c, a, torch.empty(0), short_rows=short)
    inst.b = make_rhs(inst)
    return inst


def _segment_user(inst: Instance) -> torch.Tensor:
    deg = inst.row_ptr[1:] - inst.row_ptr[:-1]
    return torch.repeat_interleave(torch.arange(inst.I, device=deg.device), deg, output_size=inst.nnz)


def make_rhs(inst: Instance) -> torch.Tensor:
    """b[j*m+k] in fp64, rounded to fp32.  "kappa": b = kappa_k * sum_i a^k_ij (BASELINE.json).
    "greedy": b = rho_jk (l_jk + eps), l = greedy load (each user sends its largest a^k_ij to that
    item), rho ~ U[0.5,1], eps = 1e-6 -- the paper's own rule for binding constraints."""
    cfg, dev = inst.cfg, inst.c.device
    J, m = cfg.J, cfg.m
    b = torch.zeros(J, m, dtype=torch.float64, device=dev)
    if cfg.rhs == "kappa":
        step = 1 << 26                                             # in pieces: config 4 has 5e9 nonzeros
        a2 = inst.a.reshape(-1, m)
        for p0 in range(0, inst.nnz, step):
            p1 = min(inst.nnz, p0 + step)
            b.index_add_(0, inst.item_idx[p0:p1].to(torch.int64), a2[p0:p1].to(torch.float64))
        b *= torch.tensor(cfg.kappa, dtype=torch.float64, device=dev)
    elif cfg.rhs == "greedy":
        a = inst.a.reshape(-1, m).to(torch.float64)
        j = inst.item_idx.to(torch.int64)
        usr = _segment_user(inst)
        for k in range(m):
            rowmax = torch.full((inst.I,), -math.inf, dtype=torch.float64, device=dev)
            rowmax.scatter_reduce_(0, usr, a[:, k], reduce="amax")
            is_max = a[:, k] == rowmax[usr]
            # ties: keep the first position in the row
            pos = torch.arange(inst.nnz, device=dev)
            firstpos = torch.full((inst.I,), inst.nnz, dtype=torch.int64, device=dev)
            firstpos.scatter_reduce_(0, usr[is_max], pos[is_max], reduce="amin")
            sel = firstpos[firstpos < inst.nnz]
            load = torch.zeros(J, dtype=torch.float64, device=dev)
            load.index_add_(0, j[sel], a[sel, k])
            rho = 0.5 + 0.5 * _uniform(cfg.seed, _S_RHO, torch.arange(J, dtype=torch.int64, device=dev) * m + k)
            b[:, k] = rho * (load + 1e-6)
    else:
        raise ValueError(cfg.rhs)
    return b.reshape(-1).to(torch.float32)


def probe_lambda(inst: Instance, which: int, lam_max: float) -> torch.Tensor:
    """Seeded lambda ~ U(0, lam_max)^{J m} in fp64 for same-lambda gradient parity probes."""
    q = torch.arange(inst.J * inst.m, dtype=torch.int64, device=inst.c.device)
    return _uniform(inst.cfg.seed + 7919 * (which + 1), _S_LAM, q) * lam_max


def perturb_c(inst: Instance, rel_std: float = 0.01) -> torch.Tensor:
    """c' = c + N(0, (rel_std*|c|)^2) i.i.d. per nonzero (config 5's drift re-solve; reading R13: std)."""
    p = torch.arange(inst.nnz, dtype=torch.int64, device=inst.c.device)
    n = _normal(inst.cfg.seed, _S_NOISE, _S_NOISE2, p)
    c64 = inst.c.to(torch.float64)
    return (c64 + rel_std * c64.abs() * n).to(torch.float32)


def proj_spec(cfg: Config):
    """(kind name, p0, p1) in the order both sides use: simplex (z,-) ; box (lo,hi) ; boxcut (ub,z)."""
    if cfg.proj == "simplex":
        return "simplex", float(cfg.proj_params[0]), 0.0
    if cfg.proj == "boxcut":
        return "boxcut", float(cfg.proj_params[0]), float(cfg.proj_params[1])
    if cfg.proj == "box":
        return "box", float(cfg.proj_params[0]), float(cfg.proj_params[1])
    raise ValueError(cfg.proj)
