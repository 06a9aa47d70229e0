"""Seeded synthetic inputs shared by the oracle-side tests and the CUDA-side
tests / bench.  Holds NONE of the method's arithmetic (no Philox, no Bezier, no
Eq. 8): only shapes, noise fields and the five BASELINE.json configurations."""
from .synth import (CONFIGS, Config, Injection, tau_linspace, noise_csd, make_sigma,  # noqa: F401
                    add_injection, config_inputs, map_seed)
