"""Seeded synthetic video-shaped Q/K/V (shared by the oracle side and the CUDA side).

Holds none of the method's arithmetic: it only draws Gaussians, scales seeded "outlier"
channel pairs and multiplies V by a library Hadamard (scipy.linalg.hadamard) — V *arrives*
Hadamard-transformed (W_v H folded offline), so this stands in for the
upstream projection, not for a step of the hot path.

Shapes and structure follow BASELINE.json `configs` and PAPER.md:L82-86 (outliers segment by
t/h/w section, sit in the low-frequency half, identical channels for Q and K).  The recipe
is restated in DESIGN.md ("Synthetic inputs").  These inputs STAND IN for the Wan2.2 /
HunyuanVideo activations the paper measures on (L190), which are not available here.
"""
from __future__ import annotations

from dataclasses import dataclass, replace

import numpy as np
from scipy.linalg import hadamard as _scipy_hadamard

SEED0 = 260702584


@dataclass(frozen=True)
class Workload:
    name: str
    cfg: int               # 1..5 (BASELINE.json configs order)
    B: int
    H: int
    D: int
    grid: tuple            # (T, Hh, W)
    n_text: int            # appended tokens without RoPE
    pairs: tuple           # (P_t, P_h, P_w)
    outlier: str           # 'tiny' | 'fixed8' | 'perhead'
    sweep_idx: int = 0

    @property
    def N(self):
        return self.grid[0] * self.grid[1] * self.grid[2] + self.n_text

    @property
    def seed(self):
        return SEED0 + 1000 * self.cfg + 10 * self.sweep_idx


TINY = Workload('tiny', 1, 1, 2, 64, (4, 8, 8), 0, (12, 10, 10), 'tiny')
WAN_1_3B = Workload('wan1.3b-480p', 2, 1, 12, 128, (21, 30, 52), 0, (22, 21, 21), 'fixed8')
WAN_14B = Workload('wan14b-720p', 3, 1, 40, 128, (21, 45, 80), 0, (22, 21, 21), 'perhead')
HUNYUAN = Workload('hunyuan', 4, 1, 24, 128, (33, 45, 80), 256, (8, 28, 28), 'perhead')
SWEEP_GRIDS = [(16, 16, 16), (16, 32, 32), (21, 30, 52), (32, 32, 64), (32, 64, 64)]
SWEEP = [Workload(f'sweep-N{g[0] * g[1] * g[2]}', 5, 1, 24, 128, g, 0, (8, 28, 28), 'perhead', i)
         for i, g in enumerate(SWEEP_GRIDS)]
ALL = {w.name: w for w in [TINY, WAN_1_3B, WAN_14B, HUNYUAN] + SWEEP}


def small_variant(w: Workload, grid, n_text=None, H=None) -> Workload:
    """Same generator on a reduced grid / head count (parity cases the oracle finishes in seconds)."""
    return replace(w, grid=tuple(grid), n_text=w.n_text if n_text is None else n_text,
                   H=w.H if H is None else H, name=w.name + '-small')


def _low_freq_half(P):
    """Section-local pair indices k >= P/2 (highest k = lowest frequency)."""
    return list(range(P // 2, P))


def outlier_spec(w: Workload, head: int):
    """-> (pair_idx[int array, global pair index], pair_scale[float array], v_chan, v_scale)."""
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([w.seed + 1, 0 if w.outlier != 'perhead' else head + 1])))
    Pt, Ph, Pw = w.pairs
    offs = [0, Pt, Pt + Ph]
    D = w.D
    if w.outlier == 'tiny':
        fixed = [offs[0] + Pt - 1, offs[1] + Ph - 1, offs[2] + Pw - 1]
        rest = [i for i in range(D // 2) if i not in fixed]
        extra = int(rng.choice(rest))
        pairs = np.array(fixed + [extra])
        scale = np.full(4, 20.0)
        vch = rng.choice(D, size=2, replace=False)
        vsc = np.full(2, 10.0)
    elif w.outlier == 'fixed8':
        loc = [[Pt - 1, Pt - 2, Pt - 3], [Ph - 1, Ph - 2, Ph - 3], [Pw - 1, Pw - 2]]
        pairs = np.array([offs[a] + k for a in range(3) for k in loc[a]])
        scale = np.full(8, 15.0)
        vch = rng.choice(D, size=4, replace=False)
        vsc = np.full(4, 8.0)
    else:
        counts = (3, 3, 2) if Pt >= 16 else (2, 3, 3)
        pl = []
        for a, P in enumerate(w.pairs):
            pl += [offs[a] + int(k) for k in rng.choice(_low_freq_half(P), size=counts[a], replace=False)]
        pairs = np.array(pl)
        scale = rng.uniform(5.0, 25.0, size=len(pairs))
        vch = rng.choice(D, size=4, replace=False)
        vsc = np.full(4, 8.0)
    return pairs, scale, np.asarray(vch), vsc


def gen_head(w: Workload, b: int, h: int):
    """fp16 Q,K (pre-RoPE) and V (Hadamard domain) of shape [N, D] for one (b,h)."""
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([w.seed, b, h])))
    N, D = w.N, w.D
    q = rng.standard_normal((N, D), dtype=np.float32)
    k = rng.standard_normal((N, D), dtype=np.float32)
    v = rng.standard_normal((N, D), dtype=np.float32)
    pairs, scale, vch, vsc = outlier_spec(w, h)
    for pidx, s in zip(pairs, scale):
        q[:, 2 * pidx:2 * pidx + 2] *= np.float32(s)
        k[:, 2 * pidx:2 * pidx + 2] *= np.float32(s)
    for c, s in zip(vch, vsc):
        v[:, c] *= np.float32(s)
    Hd = (_scipy_hadamard(D).astype(np.float32) / np.float32(np.sqrt(D)))
    v = v @ Hd
    return q.astype(np.float16), k.astype(np.float16), v.astype(np.float16)


def gen_all(w: Workload, heads=None, workers=None):
    """fp16 [B,H',N,D] for the selected heads (default all).  Every (b,h) has its own generator, so the heads are
    drawn by a small thread pool without changing any value."""
    from concurrent.futures import ThreadPoolExecutor
    heads = list(range(w.H)) if heads is None else list(heads)
    q = np.empty((w.B, len(heads), w.N, w.D), dtype=np.float16)
    k = np.empty_like(q)
    v = np.empty_like(q)

    def one(bi):
        b, i = bi
        q[b, i], k[b, i], v[b, i] = gen_head(w, b, heads[i])

    units = [(b, i) for b in range(w.B) for i in range(len(heads))]
    workers = min(8, len(units)) if workers is None else workers
    if workers <= 1:
        for u in units:
            one(u)
    else:
        with ThreadPoolExecutor(workers) as ex:
            list(ex.map(one, units))
    return q, k, v


def sample_rows(w: Workload, n_tiles=4, tile=128, head=0):
    """Seeded parity sample: n_tiles query tiles of `tile` consecutive rows (always includes the
    ragged last tile), rows clipped to N."""
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([w.seed + 2, head])))
    nt = -(-w.N // tile)
    pick = {nt - 1}
    while len(pick) < min(n_tiles, nt):
        pick.add(int(rng.integers(0, nt)))
    rows = np.concatenate([np.arange(t * tile, min(w.N, (t + 1) * tile)) for t in sorted(pick)])
    return rows
