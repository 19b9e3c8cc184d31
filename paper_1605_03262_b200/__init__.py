"""B200-native batched analytical chemical-kinetics Jacobian (arxiv 1605.03262).

`binding` is the thin ctypes layer over the C-ABI CUDA library (`include/pyjac_b200.h`);
`mechanism` / `synth` hold the model description and the seeded input generators.
"""
from .mechanism import Mechanism, MechanismBuilder  # noqa: F401

__all__ = ["Mechanism", "MechanismBuilder"]
