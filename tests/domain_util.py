"""Shared helpers of the parity tests: build seeded inputs for a config and run the oracle on it.

Inputs come from paper_1804_09101_b200.inputs (seeded generators only, no method arithmetic) evaluated on the
ORACLE's grid; the same arrays go to the oracle and to the CUDA library.
"""
from __future__ import annotations

import numpy as np

from paper_1804_09101_b200 import inputs

FIELD_SLICES = {"psi": slice(0, 10), "Pi": slice(10, 20), "Phi": slice(20, 50)}


def build_case(cfg, oracle):
    """-> (descs, coords[list of [3,P_s]], us[list of [50,P_s]], Hs[list of [4,P_s]])."""
    descs = cfg["descs"]
    coords = [oracle.coords(d) for d in descs]
    us, Hs = inputs.initial_data(descs, coords, cfg["spin"], cfg["amplitude"], cfg["id"])
    return descs, coords, us, Hs


def oracle_rhs(oracle, descs, us, Hs):
    return [oracle.rhs(d, u, H) for d, u, H in zip(descs, us, Hs)]


def field_errors(got, ref, state=None):
    """Per field X in (psi, Pi, Phi): (max |got-ref|, scale) with scale = max(||X||inf, ||ref||inf)  (reading S15).

    got/ref: [50, P] arrays of the same quantity (an RHS or a state); state: the [50, P] state the RHS was taken at
    (None when got/ref are states themselves)."""
    out = {}
    for name, sl in FIELD_SLICES.items():
        err = float(np.max(np.abs(got[sl] - ref[sl])))
        scale = float(np.max(np.abs(ref[sl])))
        if state is not None:
            scale = max(scale, float(np.max(np.abs(state[sl]))))
        out[name] = (err, scale)
    return out


def assert_parity(got, ref, state=None, tol=1e-11, what=""):
    for name, (err, scale) in field_errors(got, ref, state).items():
        assert err <= tol * scale, f"{what} field {name}: max err {err:.3e} > {tol:g} * {scale:.3e}"
