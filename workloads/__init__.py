"""Seeded synthetic inputs for the SPEAR W4A16 + gated-EC layer.

This package is the ONLY code shared by the oracle side (tests, cpu_baseline)
and the CUDA side (parity tests, bench).  It holds no arithmetic of the method
itself: it draws numbers and shapes, nothing else.  See DESIGN.md "Input
recipe" and SURVEY.md 8(d).
"""
from .synth import (  # noqa: F401
    TAGS,
    LayerInputs,
    make_layer,
    with_int8_ec,
    codes_uniform,
    normal_f64,
    uniform_f64,
    splitmix64,
)
from .configs import (  # noqa: F401
    CONFIGS,
    LayerShape,
    config_shapes,
    stack_shapes,
    algorithmic_bytes,
    algorithmic_flops,
)
