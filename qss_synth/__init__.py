"""Seeded synthetic inputs for the QSS-chemistry hot path (mechanisms and cell states).

This package is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA path
(`paper_2405_05974_b200/`). It holds no arithmetic of the method (no rate constants, no
closure, no Jacobian): it only draws random mechanisms / thermodynamic fits / cell states with
the shapes BASELINE.json prescribes (recipe: DESIGN.md "Input recipe").
The paper's real mechanisms (13-4-CH4, 35-18 n-dodecane, 55-33 n-heptane) and its
3D field are not available; these inputs stand in for them.
"""
from .mechanism import Mechanism, make_mechanism, CONFIGS, config_mechanism
from .states import make_states, make_field_states, config_states
from .toys import toy1, toy2, toy3, toy_dag, toy_nonqss
from .newton import newton_inputs, newton_inputs_torch

__all__ = [
    "Mechanism", "make_mechanism", "CONFIGS", "config_mechanism",
    "make_states", "make_field_states", "config_states",
    "toy1", "toy2", "toy3", "toy_dag", "toy_nonqss",
    "newton_inputs", "newton_inputs_torch",
]
