"""Seeded synthetic inputs for the BTA/INLA hot path.

This package holds NO arithmetic of the method (no assembly, no factorisation, no
gradient): only the model shapes of BASELINE.json's five configs, the worked example
W0, and a counter-based random generator that draws observation
sites, covariates, observations y and the hyperparameter vector theta.  Both the CPU
oracle (`oracle/`) and the CUDA path (`paper_2605_06392_b200/`) consume the arrays
produced here; neither imports the other.
"""
from .generate import (  # noqa: F401
    CONFIGS,
    EXTREME_NAMES,
    Model,
    Obs,
    make_config,
    make_w0,
    make_model,
    draw_obs,
    uniform_design,
)
