"""Seeded synthetic inputs (mechanisms and states) shared by the oracle and the CUDA
library. Holds none of the method's arithmetic; see mechanism.py / states.py."""
from .mechanism import (ELEMENTARY, THREE_BODY, LINDEMANN, TROE, P_ATM, Mechanism,
                        generate_mechanism, type_counts)
from .states import generate_states, Y_FLOOR
from .ann import KcAnn, random_kc_ann, temperature_features, RELU, ELU
from .configs import (CONFIGS, SWEEP_N, MECH_TINY, MECH_MID, MECH_LARGE, Config, MechSpec,
                      mechanism, states)

__all__ = [
    "ELEMENTARY", "THREE_BODY", "LINDEMANN", "TROE", "P_ATM", "Mechanism",
    "generate_mechanism", "type_counts", "generate_states", "Y_FLOOR", "CONFIGS",
    "SWEEP_N", "MECH_TINY", "MECH_MID", "MECH_LARGE", "Config", "MechSpec", "mechanism",
    "states", "KcAnn", "random_kc_ann", "temperature_features", "RELU", "ELU",
]
