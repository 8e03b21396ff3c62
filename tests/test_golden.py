"""Golden fixtures (tests/golden/): values fixed by the mathematics, not by the oracle (CPU only)."""
import math
import os

import numpy as np
import pytest

from oracle import Oracle
from tpc_synth import default_params, generate_config

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _rows(name):
    with open(os.path.join(GOLDEN, name)) as f:
        return [tuple(float(v) for v in ln.split()) for ln in f if ln.strip() and not ln.startswith("#")]


@pytest.mark.parametrize("pt,bz,radius", _rows("helix_radius.txt"))
def test_helix_step_follows_the_textbook_radius(pt, bz, radius):
    """A track starting parallel to x (sin(phi) = 0) at distance dx along x has sin(phi) = dx / R and has moved
    sideways by the sagitta R - sqrt(R^2 - dx^2); arc length R * asin(dx / R) gives z through tan(lambda)."""
    tf = generate_config("cfg1")
    P = default_params(tf)
    P["bz_tesla"] = np.float32(bz)
    o = Oracle(P)
    dx, tanl = 4.0, 0.7
    for charge in (+1.0, -1.0):
        ok, p1, _, _ = o.kf_propagate([0.0, 0.0, 0.0, tanl, charge / pt], np.zeros(15), 100.0, 100.0 + dx, precision=64)
        assert ok
        assert math.isclose(abs(p1[2]), dx / radius, rel_tol=2e-7)      # kb is one fp32 product (section 3.0)
        assert math.isclose(abs(p1[0]), radius - math.sqrt(radius * radius - dx * dx), rel_tol=1e-6)
        assert math.isclose(p1[1], tanl * radius * math.asin(dx / radius), rel_tol=1e-9)
        assert np.sign(p1[2]) == -charge       # kb < 0 for Bz > 0 (DESIGN.md 3.6 #12; the generator uses the same sign)
