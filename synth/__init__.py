"""Seeded synthetic pCT inputs (phantoms + tracker histories) that serve BOTH the oracle tests and
the CUDA path's tests/bench.  Holds none of the method's arithmetic (no hull, MLP, walk or DROP):
it is the *forward* model that stands in for the scanner data the paper used,
following the recipe in DESIGN.md "Synthetic inputs"."""
from .phantoms import Config, config, rsp_at, rsp_volume  # noqa: F401
from .generate import generate_numpy, FIELDS  # noqa: F401
