"""Seeded synthetic jets shaped like the paper's workload (<= 100 particles x
(features + 2 coordinates + mask), fp32, pseudo-random inputs).  Recipes follow BASELINE.json `configs` and the
readings R23-R25 of DESIGN.md.  Ragged layout: particle-major rows, jets contiguous, int32 CSR offsets.
"""
from dataclasses import dataclass
import numpy as np


@dataclass
class JetBatch:
    feats: np.ndarray     # [N, F] fp32
    coords: np.ndarray    # [N, 2] fp32
    offsets: np.ndarray   # [B+1] int32

    @property
    def n_jets(self) -> int:
        return int(self.offsets.size - 1)

    @property
    def n_particles(self) -> int:
        return int(self.offsets[-1])

    def counts(self) -> np.ndarray:
        return np.diff(self.offsets)

    def head(self, b: int) -> "JetBatch":
        """First b jets (config 5: nested batch sizes)."""
        n = int(self.offsets[b])
        return JetBatch(self.feats[:n].copy(), self.coords[:n].copy(), self.offsets[:b + 1].copy())

    def select(self, jets) -> "JetBatch":
        jets = list(jets)
        f = [self.feats[self.offsets[j]:self.offsets[j + 1]] for j in jets]
        c = [self.coords[self.offsets[j]:self.offsets[j + 1]] for j in jets]
        return _pack(f, c, self.feats.shape[1])


def _pack(feats, coords, F) -> JetBatch:
    cnt = np.array([len(f) for f in feats], dtype=np.int64)
    off = np.zeros(len(feats) + 1, dtype=np.int32)
    off[1:] = np.cumsum(cnt)
    if len(feats) and off[-1] > 0:
        f = np.concatenate([np.asarray(x, dtype=np.float64).reshape(-1, F) for x in feats]).astype(np.float32)
        c = np.concatenate([np.asarray(x, dtype=np.float64).reshape(-1, 2) for x in coords]).astype(np.float32)
    else:
        f = np.zeros((0, F), np.float32)
        c = np.zeros((0, 2), np.float32)
    return JetBatch(np.ascontiguousarray(f), np.ascontiguousarray(c), off)


def _project(c, rmax=0.8):
    """R23: radial projection onto r <= rmax (no resampling, so RNG consumption is fixed)."""
    r = np.sqrt((c ** 2).sum(1))
    s = np.where(r > rmax, rmax / np.maximum(r, 1e-300), 1.0)
    return c * s[:, None]


def _kin_features(c, pt):
    """R24: [ln pT, ln E, ln pT-rel, ln E-rel, dR, eta, phi], E = pT cosh(eta)."""
    e = pt * np.cosh(c[:, 0])
    return np.stack([np.log(pt), np.log(e), np.log(pt / pt.sum()), np.log(e / e.sum()),
                     np.sqrt((c ** 2).sum(1)), c[:, 0], c[:, 1]], axis=1)


def make_tiny(seed: int = 1001, n_jets: int = 32, n: int = 16, F: int = 4) -> JetBatch:
    """configs[0]: exactly 16 particles, coords ~ N(0,0.2) projected to r<=0.8, 4 features ~ N(0,1)."""
    rng = np.random.default_rng(seed)
    fs, cs = [], []
    for _ in range(n_jets):
        c = _project(rng.normal(0.0, 0.2, (n, 2)))
        f = rng.normal(0.0, 1.0, (n, F))
        fs.append(f); cs.append(c)
    return _pack(fs, cs, F)


def _physics_jets(rng, n_jets, lam, nmin, nmax, extra):
    fs, cs = [], []
    for _ in range(n_jets):
        n = int(np.clip(rng.poisson(lam), nmin, nmax))
        c = _project(rng.normal(0.0, 0.2, (n, 2)))
        pt = rng.lognormal(1.0, 1.0, n)
        f = _kin_features(c, pt)
        if extra:
            f = np.concatenate([f, rng.normal(0.0, 1.0, (n, extra))], axis=1)   # R25
        fs.append(f); cs.append(c)
    return _pack(fs, cs, 7 + extra)


def make_particlenet_batch(seed: int = 1002, n_jets: int = 1024, nmax: int = 100) -> JetBatch:
    """configs[1]: multiplicity ~ clip(Poisson(40),5,100), 7 kinematic features."""
    return _physics_jets(np.random.default_rng(seed), n_jets, 40, 5, nmax, 0)


def make_paper_f5_batch(seed: int = 1002, n_jets: int = 1024, nmax: int = 100) -> JetBatch:
    """The paper-literal input width ("five input features"): the configs[1] jets with their first five
    feature columns (log pT, log E, log pT-rel, log E-rel, dR); the paper does not name its five."""
    b = make_particlenet_batch(seed=seed, n_jets=n_jets, nmax=nmax)
    return JetBatch(np.ascontiguousarray(b.feats[:, :5]), b.coords, b.offsets)


def to_channel_first(feats, coords, mask):
    """[B, P, F], [B, P, 2], [B, P] -> the served model's tensors: points [B, 2, P], features [B, F, P],
    mask [B, 1, P]; a pure relayout."""
    return (np.ascontiguousarray(np.transpose(coords, (0, 2, 1))), np.ascontiguousarray(np.transpose(feats, (0, 2, 1))),
            np.ascontiguousarray(mask[:, None, :]))


def make_ragged_batch(seed: int = 1003, n_jets: int = 4096) -> JetBatch:
    """configs[2]: clip(Poisson(40),5,128), 9 features (7 kinematic + 2 ~ N(0,1))."""
    return _physics_jets(np.random.default_rng(seed), n_jets, 40, 5, 128, 2)


def make_sweep_batch(seed: int = 1005, n_jets: int = 16384) -> JetBatch:
    """configs[4]: clip(Poisson(60),5,128), 7 features; batch size B uses the first B jets."""
    return _physics_jets(np.random.default_rng(seed), n_jets, 60, 5, 128, 0)


def make_client_pool(client: int, n_requests: int = 64, jets_per_request: int = 16):
    """configs[3]: client c pre-generates a pool of requests of 16 jets (config-2 jet recipe), seed 1004*100+c."""
    rng = np.random.default_rng(1004 * 100 + client)
    return [_physics_jets(rng, jets_per_request, 40, 5, 100, 0) for _ in range(n_requests)]


def make_edge_case_batch(F: int, seed: int = 77, sizes=(0, 1, 2, 3, 5, 16, 17, 18, 100, 127, 128, 0, 40),
                         scale: float = 1.0) -> JetBatch:
    """Degenerate multiplicities (DESIGN.md edge-case set): n = 0, 1, n-1 < k, n = k+1, max sizes."""
    rng = np.random.default_rng(seed)
    fs, cs = [], []
    for n in sizes:
        cs.append(_project(rng.normal(0.0, 0.2, (n, 2))))
        fs.append(rng.normal(0.0, scale, (n, F)))
    return _pack(fs, cs, F)


def pad_batch(b: JetBatch, P: int, seed: int = 5, interleave: bool = False, garbage=np.nan):
    """Padded form [B,P,F], [B,P,2], mask [B,P] (features, coordinates, mask).  Masked slots hold
    `garbage`; with interleave=True real particles sit at random slots in their original relative order."""
    B, F = b.n_jets, b.feats.shape[1]
    rng = np.random.default_rng(seed)
    feats = np.full((B, P, F), garbage, np.float32)
    coords = np.full((B, P, 2), garbage, np.float32)
    mask = np.zeros((B, P), np.float32)
    for j in range(B):
        s, e = int(b.offsets[j]), int(b.offsets[j + 1])
        n = e - s
        assert n <= P
        slots = np.sort(rng.choice(P, n, replace=False)) if interleave else np.arange(n)
        feats[j, slots] = b.feats[s:e]
        coords[j, slots] = b.coords[s:e]
        mask[j, slots] = 1.0
    return feats, coords, mask
