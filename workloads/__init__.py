"""Seeded synthetic inputs for the SOAP disk-integration hot path.

This package holds the input generators only.  It contains none of the method's
arithmetic (no Doppler shift, no interpolation, no disk geometry): it builds the
*inputs* the method consumes - wavelength-grid parameters, mu-binned quiet / spot /
facula spectra, contrast arrays, active-region lists and phases - with the shapes
and structure of the paper's workloads, which were
measured on solar atlases that are not available here.

Both the CPU oracle's tests and the CUDA path's tests/bench draw their inputs from
here; neither of those two imports the other.
"""
from .synth import (  # noqa: F401
    Workload,
    make_workload,
    make_config1,
    make_config2,
    make_config3,
    make_config4,
    make_config5_star,
    CONFIG_NAMES,
    evolution_radii,
    SEED_BASE,
)
