"""Seeded synthetic inputs for the chemistry step (G1-G3, G6, G7).

This module serves both the CUDA path and the oracle and therefore holds NONE of the method's
arithmetic: it only draws random numbers with the shapes, ranges and structure of the paper's
workloads (LES cell fields at ~1 atm with mass fractions spanning many decades, PAPER.md:98, 148;
a DRM19-sized mechanism; an MLP with hidden layers 1600-800-400).
The derived inputs -- the conserved enthalpy h(T, Y) (G5) and the input normalisation statistics
over [T, p, F(Y)] (G4) -- need the NASA-7 polynomials and the Box-Cox transform, so they are NOT
computed here: tests take them from oracle/, bench.py from the library's own helper calls
(gpuann_enthalpy, gpuann_input_moments).

They stand in for the paper's LES fields, DRM19 thermo data and trained weights, none of which exist here.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional, Tuple

import numpy as np

P_ATM = 101325.0


@dataclass(frozen=True)
class Config:
    """One of BASELINE.json `configs[0..4]`."""
    name: str
    index: int
    n_cells: int
    n_species: int
    hidden: Tuple[int, ...]
    precision: int              # 0 = FP32 CUDA-core path, 1 = BF16 tcgen05 path, 2 = FP16 tcgen05 path
    dt: float = 1e-6            # delta t = 1 us
    newton_max_iter: int = 20
    newton_tol: float = 1e-6
    T_active: float = 0.0       # <= 0: all cells active
    mixed_field: bool = False   # G6 (configs[4])
    lam: float = 0.1
    sigma_out: float = 2.0e4    # 1/s, G4
    T_min: float = 200.0
    T_max: float = 3500.0

    @property
    def sizes(self) -> Tuple[int, ...]:
        return (2 + self.n_species,) + tuple(self.hidden) + (self.n_species,)

    @property
    def flop_per_cell(self) -> int:
        s = self.sizes
        return 2 * sum(s[i] * s[i + 1] for i in range(len(s) - 1))

    @property
    def state_bytes_per_cell(self) -> int:
        return (3 + self.n_species) * 4 + (1 + self.n_species) * 4


CONFIGS: List[Config] = [
    Config("c0", 0, 4096, 9, (64, 64), precision=0),
    Config("c1", 1, 65536, 21, (400, 200, 100), precision=1),
    Config("c2", 2, 1048576, 21, (1600, 800, 400), precision=1),
    Config("c3", 3, 4194304, 36, (1600, 800, 400), precision=1, dt=5e-7, newton_max_iter=10),
    Config("c4", 4, 8388608, 21, (1600, 800, 400), precision=1, T_active=600.0, mixed_field=True),
]
# configs[1] / configs[2] in the half precision the paper itself infers in: same
# seeds, states and FP32 draws; the weights are rounded to FP16 instead of BF16.  Not BASELINE.json configs (index kept).
VARIANTS: List[Config] = [
    Config("c1h", 1, 65536, 21, (400, 200, 100), precision=2),
    Config("c2h", 2, 1048576, 21, (1600, 800, 400), precision=2),
]


def get_config(name_or_index) -> Config:
    for c in CONFIGS:
        if c.name == name_or_index or c.index == name_or_index:
            return c
    for c in VARIANTS:
        if c.name == name_or_index:
            return c
    raise KeyError(name_or_index)


@dataclass
class State:
    T: np.ndarray   # [n] f32, K
    p: np.ndarray   # [n] f32, Pa
    Y: np.ndarray   # [Ns][n] f32, species-major


@dataclass
class Thermo:
    nasa_lo: np.ndarray          # [Ns][7] f64
    nasa_hi: Optional[np.ndarray]  # None = one range
    T_mid: Optional[np.ndarray]
    W: np.ndarray                # [Ns] f64 kg/kmol


@dataclass
class Net:
    sizes: Tuple[int, ...]
    weights: List[np.ndarray]    # [out][in] f32 (BF16-representable if rounded)
    biases: List[np.ndarray]     # [out] f32


def round_to_bf16(a: np.ndarray) -> np.ndarray:
    """Round FP32 values to the nearest BF16-representable value (ties to even); result stays FP32."""
    a = np.ascontiguousarray(a, dtype=np.float32)
    u = a.view(np.uint32).astype(np.uint64)
    lsb = (u >> 16) & 1
    u = (u + 0x7FFF + lsb) & 0xFFFF0000
    return u.astype(np.uint32).view(np.float32).reshape(a.shape)


def gen_state(rng: np.random.Generator, n: int, Ns: int) -> State:
    """G1: T ~ U[300, 2500] K, p = 101325 * U[0.95, 1.05] Pa, Y ~ Dirichlet(0.5)."""
    T = rng.uniform(300.0, 2500.0, n)
    p = P_ATM * rng.uniform(0.95, 1.05, n)
    Y = rng.dirichlet(0.5 * np.ones(Ns), n).T
    return State(T.astype(np.float32), p.astype(np.float32), np.ascontiguousarray(Y, dtype=np.float32))


def fresh_composition(Ns: int) -> np.ndarray:
    """G6: fixed fresh-mixture vector, placed by index (a stoichiometric methane/air-like split)."""
    y = np.zeros(Ns)
    y[0], y[1], y[Ns - 1] = 0.055, 0.220, 0.725
    return y


def gen_mixed_state(rng: np.random.Generator, n: int, Ns: int) -> State:
    """G6 (configs[4]): 70 % near-fresh cells, 30 % flame cells, shuffled by the seed."""
    n_f = int(round(0.7 * n))
    n_b = n - n_f
    T_f = rng.uniform(300.0, 700.0, n_f)
    Y_f = fresh_composition(Ns)[None, :] + rng.normal(0.0, 1e-4, (n_f, Ns))
    Y_f = np.maximum(Y_f, 0.0)
    Y_f = Y_f / Y_f.sum(axis=1, keepdims=True)
    T_b = rng.uniform(1200.0, 2400.0, n_b)
    Y_b = rng.dirichlet(0.5 * np.ones(Ns), n_b)
    p = P_ATM * rng.uniform(0.95, 1.05, n)
    perm = rng.permutation(n)
    T = np.concatenate([T_f, T_b])[perm]
    Y = np.concatenate([Y_f, Y_b], axis=0)[perm]
    return State(T.astype(np.float32), p.astype(np.float32), np.ascontiguousarray(Y.T, dtype=np.float32))


def gen_thermo(rng: np.random.Generator, Ns: int) -> Thermo:
    """G2: synthetic NASA-7 coefficients, one range 200-3500 K, molar masses U[2, 44] kg/kmol."""
    a = np.zeros((Ns, 7))
    a[:, 0] = rng.uniform(2.5, 4.5, Ns)
    a[:, 1] = rng.uniform(0.0, 2e-3, Ns)
    a[:, 2] = rng.uniform(-1e-7, 0.0, Ns)
    a[:, 5] = rng.uniform(-3e4, 3e4, Ns)
    W = rng.uniform(2.0, 44.0, Ns)
    return Thermo(a, None, None, W)


def gen_net(rng: np.random.Generator, sizes, bf16_weights: bool, f16_weights: bool = False) -> Net:
    """G3: Xavier-uniform weights, U[-1/sqrt(fan_in), 1/sqrt(fan_in)] biases, layer by layer."""
    ws, bs = [], []
    for l in range(len(sizes) - 1):
        fan_in, fan_out = sizes[l], sizes[l + 1]
        a = np.sqrt(6.0 / (fan_in + fan_out))
        w = rng.uniform(-a, a, (fan_out, fan_in)).astype(np.float32)
        b = rng.uniform(-1.0 / np.sqrt(fan_in), 1.0 / np.sqrt(fan_in), fan_out).astype(np.float32)
        if bf16_weights:
            w = round_to_bf16(w)
        if f16_weights:
            w = w.astype(np.float16).astype(np.float32)   # round to nearest even
        ws.append(w)
        bs.append(b)
    return Net(tuple(sizes), ws, bs)


@dataclass
class Problem:
    cfg: Config
    n: int
    state: State
    thermo: Thermo
    net: Net
    out_mean: np.ndarray  # [Ns] f32
    out_std: np.ndarray   # [Ns] f32


def make_problem(cfg: Config, n: Optional[int] = None, seed: Optional[int] = None) -> Problem:
    """Draws, strictly in this order: state (G1 or G6), thermo (G2), net (G3).  seed defaults to cfg.index."""
    n = cfg.n_cells if n is None else int(n)
    rng = np.random.default_rng(cfg.index if seed is None else seed)
    Ns = cfg.n_species
    state = gen_mixed_state(rng, n, Ns) if cfg.mixed_field else gen_state(rng, n, Ns)
    thermo = gen_thermo(rng, Ns)
    net = gen_net(rng, cfg.sizes, bf16_weights=(cfg.precision == 1), f16_weights=(cfg.precision == 2))
    out_mean = np.zeros(Ns, dtype=np.float32)
    out_std = np.full(Ns, cfg.sigma_out, dtype=np.float32)
    return Problem(cfg, n, state, thermo, net, out_mean, out_std)


def gen_ensemble(cfg: Config, seed: int):
    """SURVEY.md 8(f) NEXT-1 / PAPER.md:103: Ns nets of the shape `D - hidden... - 1` drawn like G3 (Xavier-uniform weights,
    U[+-1/sqrt(fan_in)] biases, net after net from one generator), rounded like the config's single net.  Returns
    (sizes, weights[k][l], biases[k][l])."""
    rng = np.random.default_rng(seed)
    sizes = (2 + cfg.n_species,) + tuple(cfg.hidden) + (1,)
    nets = [gen_net(rng, sizes, bf16_weights=(cfg.precision == 1), f16_weights=(cfg.precision == 2)) for _ in range(cfg.n_species)]
    return sizes, [n.weights for n in nets], [n.biases for n in nets]
