"""Seeded synthetic inputs for the plane-wave H|psi> path (BASELINE.json `configs`).

This package is *input data only*.  It is used by the oracle tests, the GPU
parity tests and bench.py alike, and by design holds none of the method's
arithmetic: no sphere construction, no kinetic energies, no FFT of psi, no
projector evaluation.  Quantities that depend on the method (the `kin` array
that shapes the psi envelope) are passed in by the caller.

Recipe: SURVEY.md section 8(d) "Synthetic inputs" restating BASELINE.json.
"""
from .rng import normals, uniforms            # noqa: F401
from .cells import (CONFIG_NAMES, make_config, gen_psi, gen_psi_band, gen_psi_torch,   # noqa: F401
                    config_seed, projector_l, gamma_dij, spinor_inputs, gen_vloc)
