"""Seeded synthetic workloads for the DASH 4D hash encoder (G_4D).

This module is the ONLY thing the oracle side (`oracle/`, `tests/`) and the CUDA side
(`paper_2507_19141_b200/`, `bench.py`) have in common.  It holds none of the method's
arithmetic: no resolution schedule, no hashing, no interpolation — only
  * the encoder hyper-parameters of BASELINE.json's five configs as plain numbers, and
  * numpy PCG64 draws of queries, tables and upstream gradients (recipe: DESIGN.md §4,
    SURVEY.md §8d / Q18-Q20).

The inputs stand in for the paper's workloads, which are not available offline: Neural 3D
Video has 300 frames per scene, coffee-martini trains ~106.6k Gaussians
(PAPER.md:229), dynamic regions are spatially clustered (Fig. 7).

Draw order per config (fixed; changing it changes every expected value):
    centres, cluster ids, normals  -> xyz        (C1: one (N,4) uniform draw instead)
    t
    [permutation]                                (C5 only)
    table
    dY
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

# largest fp32 below 1: inputs are clamped into [0, 1 - 2^-24] (reading Q12/Q19)
ONE_MINUS_EPS = np.float32(1.0) - np.float32(2.0 ** -24)


@dataclass(frozen=True)
class EncoderParams:
    """Hyper-parameters of G_4D: L levels, F features, T entries per level,
    geometric resolution ranges for (x,y,z) and for t.  table_dtype: 'fp32' or 'fp16'."""
    L: int
    F: int
    T: int
    res_s_min: int
    res_s_max: int
    res_t_min: int
    res_t_max: int
    table_dtype: str = "fp32"


@dataclass(frozen=True)
class WorkloadSpec:
    name: str
    seed: int
    N: int                      # number of queries
    enc: EncoderParams
    kind: str                   # 'uniform' | 'clustered'
    clusters: int = 0
    sigma: float = 0.0
    t_kind: str = "uniform"     # 'uniform' | 'frames300'
    rows: int = 0               # C5: M xyz rows (0 => rows == N, no index list)
    selected: int = 0           # C5: rows marked dynamic
    repeats: int = 1            # C5: timestamps per dynamic row
    note: str = ""


CONFIGS = {
    # BASELINE.json configs[0..4]; seeds: config i uses seed i-1
    "C1": WorkloadSpec("C1", 0, 4096, EncoderParams(4, 2, 1 << 12, 16, 128, 8, 32), "uniform",
                       note="tiny: xyzt iid U[0,1)^4"),
    "C2": WorkloadSpec("C2", 1, 100_000, EncoderParams(16, 2, 1 << 17, 16, 2048, 8, 150), "clustered",
                       clusters=64, sigma=0.05, t_kind="frames300"),
    "C3": WorkloadSpec("C3", 2, 300_000, EncoderParams(16, 2, 1 << 19, 16, 4096, 8, 300), "clustered",
                       clusters=64, sigma=0.05, t_kind="frames300"),
    "C4": WorkloadSpec("C4", 3, 1_000_000, EncoderParams(16, 4, 1 << 21, 16, 4096, 8, 300, "fp16"),
                       "clustered", clusters=256, sigma=0.02, t_kind="uniform"),
    "C5": WorkloadSpec("C5", 4, 1_800_000, EncoderParams(16, 2, 1 << 19, 16, 4096, 8, 300), "clustered",
                       clusters=64, sigma=0.05, t_kind="uniform",
                       rows=1_500_000, selected=450_000, repeats=4,
                       note="training-step shape: int32 index list into 1.5M rows, 4 timestamps each"),
}


@dataclass
class Workload:
    spec: WorkloadSpec
    xyz: np.ndarray                 # [rows][3] fp32, C-contiguous
    t: np.ndarray                   # [N] fp32
    index: Optional[np.ndarray]     # [N] int32 or None
    table: Optional[np.ndarray] = None   # [L][T][F] fp32 or fp16
    dout: Optional[np.ndarray] = None    # [N][L*F] fp32
    meta: dict = field(default_factory=dict)

    @property
    def N(self) -> int:
        return int(self.t.shape[0])


def _clustered_xyz(rng: np.random.Generator, n: int, clusters: int, sigma: float) -> np.ndarray:
    centres = rng.uniform(0.15, 0.85, size=(clusters, 3))             # float64
    ids = rng.integers(0, clusters, size=n)
    normals = rng.standard_normal(size=(n, 3))
    xyz = centres[ids] + sigma * normals
    xyz = np.clip(xyz, 0.0, None).astype(np.float32)
    return np.minimum(xyz, ONE_MINUS_EPS)                              # clamp, not reject (Q19)


def make_table(rng: np.random.Generator, enc: EncoderParams) -> np.ndarray:
    """iid U(-1e-4, 1e-4) (BASELINE.json config 1; used for every config, reading Q18).
    fp16 tables are the fp32 draw rounded to half once, on the host."""
    tab = rng.uniform(-1e-4, 1e-4, size=(enc.L, enc.T, enc.F)).astype(np.float32)
    if enc.table_dtype == "fp16":
        tab = tab.astype(np.float16)
    return tab


def make_workload(name: str, *, n_override: Optional[int] = None, with_table: bool = True,
                  with_dout: bool = True) -> Workload:
    """Build config `name` ('C1'..'C5').  n_override shrinks the query count (and, for C5, the
    row/selection counts in proportion) while keeping distribution and encoder parameters —
    used for bounded oracle samples; the draw order is unchanged."""
    spec = CONFIGS[name]
    enc = spec.enc
    rng = np.random.default_rng(spec.seed)
    N = spec.N if n_override is None else int(n_override)
    index = None
    if spec.kind == "uniform":
        q = rng.random(size=(N, 4), dtype=np.float32)                  # [0,1), multiples of 2^-24
        xyz = np.ascontiguousarray(q[:, :3])
        t = np.ascontiguousarray(q[:, 3])
    else:
        if spec.rows:
            scale = N / spec.N
            rows = max(1, int(round(spec.rows * scale)))
            selected = max(1, N // spec.repeats)
            N = selected * spec.repeats
        else:
            rows, selected = N, 0
        xyz = _clustered_xyz(rng, rows, spec.clusters, spec.sigma)
        if spec.t_kind == "frames300":
            j = rng.integers(0, 300, size=N)
            t = (j.astype(np.float64) / 300.0).astype(np.float32)      # frame-aligned timestamps
        else:
            t = rng.random(size=N, dtype=np.float32)
        if spec.rows:
            perm = rng.permutation(rows)
            chosen = np.sort(perm[:selected]).astype(np.int32)         # what nonzero(mask) yields
            index = np.repeat(chosen, spec.repeats).astype(np.int32)   # each id 4x, consecutive
    w = Workload(spec, xyz, t, index)
    if with_table:
        w.table = make_table(rng, enc)
    if with_dout:
        w.dout = rng.standard_normal(size=(N, enc.L * enc.F), dtype=np.float32)
    return w


def make_queries_uniform(seed: int, n: int) -> tuple[np.ndarray, np.ndarray]:
    """Small helper for tests: n iid uniform queries, (xyz [n][3], t [n])."""
    rng = np.random.default_rng(seed)
    q = rng.random(size=(n, 4), dtype=np.float32)
    return np.ascontiguousarray(q[:, :3]), np.ascontiguousarray(q[:, 3])


def make_points_clustered(seed: int, n: int, clusters: int = 64, sigma: float = 0.05) -> np.ndarray:
    """n points [n][3] fp32 from the clustered recipe of C2-C5 (centres U[0.15,0.85]^3, Gaussian blobs,
    clamped) — the Gaussian centres p that the 3D encoder G_3D of the decomposition stage sees
    (ALL Gaussians, static and dynamic)."""
    return np.ascontiguousarray(_clustered_xyz(np.random.default_rng(seed), n, clusters, sigma))


# G_3D workload for bench extras / full-size parity: the 1.5M Gaussians of C5's scene through an
# Instant-NGP-sized 3D encoder (the paper gives no G_3D hyper-parameters; Q26).
G3D_SPEC = WorkloadSpec("G3D", 5, 1_500_000, EncoderParams(16, 2, 1 << 19, 16, 2048, 1, 1), "clustered",
                        clusters=64, sigma=0.05, note="decomposition stage: every Gaussian, no timestamp")


def make_g3d_workload(n_override: Optional[int] = None) -> Workload:
    spec = G3D_SPEC
    rng = np.random.default_rng(spec.seed)
    N = spec.N if n_override is None else int(n_override)
    xyz = _clustered_xyz(rng, N, spec.clusters, spec.sigma)
    w = Workload(spec, xyz, np.zeros(N, np.float32), None)
    w.table = make_table(rng, spec.enc)
    w.dout = rng.standard_normal(size=(N, spec.enc.L * spec.enc.F), dtype=np.float32)
    return w


def make_mlp_params(seed: int, widths) -> np.ndarray:
    """Packed fp32 parameters [W_1 | b_1 | W_2 | b_2 | ...] of a dense-layer chain (phi_d + heads, PAPER.md:133-142;
    sizes are not in the paper): W_l, b_l iid U(-1/sqrt(K_l), 1/sqrt(K_l)), K_l the layer's input width — the
    default initialisation of a linear layer, so activations keep the scale of the features."""
    rng = np.random.default_rng(seed)
    parts = []
    for l in range(1, len(widths)):
        k = 1.0 / np.sqrt(widths[l - 1])
        parts.append(rng.uniform(-k, k, size=widths[l] * widths[l - 1]))
        parts.append(rng.uniform(-k, k, size=widths[l]))
    return np.concatenate(parts).astype(np.float32)
