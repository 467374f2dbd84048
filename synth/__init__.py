"""Seeded synthetic pCT inputs (phantoms + tracker histories) that serve BOTH the oracle tests and
the CUDA path's tests/bench.  Holds none of the method's arithmetic (no hull, MLP, walk or DROP):
it is the *forward* model that stands in for the scanner data the paper used,
following the recipe in DESIGN.md "Synthetic inputs"."""
from .phantoms import Config, config, rsp_at, rsp_volume  # noqa: F401
from .generate import generate_numpy, FIELDS  # noqa: F401

# names of the arrays in include/pct.h, keyed by this package's beam-frame names (no arithmetic)
PCT_NAMES = dict(t_in="entry_t", v_in="entry_v", t_out="exit_t", v_out="exit_v", tht_in="entry_dt",
                 thv_in="entry_dv", tht_out="exit_dt", thv_out="exit_dv", wepl="wepl", proj="proj",
                 proj_cos="proj_cos", proj_sin="proj_sin")


def to_pct_names(arrays):
    """Re-key a generated dict (numpy arrays or CUDA tensors) with the field names of include/pct.h."""
    return {PCT_NAMES[k]: v for k, v in arrays.items()}
