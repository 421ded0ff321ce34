"""The five workloads of BASELINE.json `configs`, as seeds + shapes (inputs only).

Seeds follow SURVEY.md section 8(d): mechanism seeds 9/21 -> 2008, 53/325 -> 8483,
111/784 -> 20088483; state seed = mechanism seed + 1000 * config index.
"""
from __future__ import annotations

import dataclasses
import functools

from .mechanism import Mechanism, generate_mechanism
from .states import generate_states

ELEMENTS_3 = ("H", "O", "N")
ELEMENTS_5 = ("C", "H", "O", "N", "Ar")


@dataclasses.dataclass(frozen=True)
class MechSpec:
    name: str
    S: int
    R: int
    elements: tuple
    seed: int
    frac_three_body: float
    frac_falloff: float


@dataclasses.dataclass(frozen=True)
class Config:
    name: str
    mech: MechSpec
    N: int
    state_seed: int
    T_range: tuple
    P_range_atm: tuple
    dirichlet_alpha: float


MECH_TINY = MechSpec("S9_R21", 9, 21, ELEMENTS_3, 2008, 0.20, 0.10)
MECH_MID = MechSpec("S53_R325", 53, 325, ELEMENTS_5, 8483, 0.30, 0.08)
MECH_LARGE = MechSpec("S111_R784", 111, 784, ELEMENTS_5, 20088483, 0.25, 0.10)

CONFIGS = {
    # configs[0]: tiny mechanism, the case the oracle finishes in no time
    "tiny_1k": Config("tiny_1k", MECH_TINY, 1024, 2008 + 1000, (1000.0, 2500.0), (1.0, 10.0), 1.0),
    # configs[1]: same generator, throughput run in the small-mechanism regime
    "tiny_1m": Config("tiny_1m", MECH_TINY, 1 << 20, 2008 + 2000, (1000.0, 2500.0), (1.0, 10.0), 1.0),
    # configs[2]: the configuration BASELINE.json's metric is quoted on
    "mid_1m": Config("mid_1m", MECH_MID, 1 << 20, 8483 + 3000, (900.0, 2800.0), (1.0, 40.0), 0.5),
    # configs[3]: large mechanism
    "large_256k": Config("large_256k", MECH_LARGE, 1 << 18, 20088483 + 4000, (900.0, 2800.0), (1.0, 40.0), 0.5),
    # configs[4] RK4 part: 65536 independent cells, T0 ~ U[1100, 1500] K
    "mid_rk4": Config("mid_rk4", MECH_MID, 65536, 8483 + 5000, (1100.0, 1500.0), (1.0, 40.0), 0.5),
}

# configs[4] sweep part: N = 2^8, 2^10, ..., 2^22 at S=53/R=325, config-3 state distribution
SWEEP_N = tuple(1 << e for e in range(8, 23, 2))


@functools.lru_cache(maxsize=8)
def mechanism(spec: MechSpec) -> Mechanism:
    return generate_mechanism(spec.S, spec.R, spec.elements, spec.seed,
                              spec.frac_three_body, spec.frac_falloff)


def states(cfg: Config, N=None, seed_offset=0):
    """States for `cfg`; N overrides the config's cell count (sweeps, samples)."""
    n = cfg.N if N is None else int(N)
    return generate_states(cfg.mech.S, n, cfg.state_seed + seed_offset, cfg.T_range,
                           cfg.P_range_atm, cfg.dirichlet_alpha)
