"""FP64 CPU oracle for the GPU-ANN chemistry step -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It imports nothing from paper_2402_18858_b200 (and vice versa).
"""
from .oracle import (  # noqa: F401
    Oracle,
    OracleDerived,
    OracleModel,
    boxcox,
    boxcox_inv,
    build,
    enthalpy_field,
    gelu,
    input_moments,
    mixture_cp,
    mixture_h,
    mlp_forward,
    newton_T,
    num_threads,
    set_num_threads,
    species_cp,
    species_h,
)
