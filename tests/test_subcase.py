"""CPU check of the premise of the full-size GPU parity test: the oracle evaluated on the two-ring neighbourhood of sampled elements
(tests/gpu_util.subcase) reproduces the full-mesh oracle at those elements -- Euler needs one ring, Navier-Stokes two."""
import numpy as np
import pytest

from fr_inputs import cases
from gpu_util import subcase
from util import oracle_rhs


@pytest.mark.parametrize("system,rings,exact", [("ns", 2, True), ("euler", 1, True), ("ns", 1, False)])
def test_subcase_oracle_equals_full_oracle_at_seeds(system, rings, exact):
    case = cases.config3(p=2, ntheta=16, nz=3, nlayers=4, nr=4, numbering="random", system=system)
    full = oracle_rhs(case)
    rng = np.random.Generator(np.random.PCG64(7))
    seeds = []
    for t, e in enumerate(case["eles"]):
        s = list(rng.integers(0, e["neles"], 6)) + [0, e["neles"] - 1]
        for b in case["bcs"]:
            on = b["ele"][b["et"] == t]
            if len(on):
                s += list(on[:2])
        seeds.append(np.unique(np.array(s, dtype=np.int64)))
    sub, pos = subcase(case, seeds, rings=rings)
    assert all(se["neles"] < e["neles"] for se, e in zip(sub["eles"], case["eles"]))
    ref = oracle_rhs(sub)
    err = 0.0
    for t in range(len(seeds)):
        a, b = full[t][:, :, seeds[t]], ref[t][:, :, pos[t]]
        err = max(err, np.abs(a - b).max() / np.abs(a).max())
    if exact:
        assert err < 1e-12, err
    else:
        assert err > 1e-6, err      # one ring is not enough for the viscous terms: the test would notice a too-small halo
