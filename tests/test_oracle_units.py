"""Pins for the physical-units front end (device of ref. [42])."""
import math

import pytest

from oracle import units as ou
from paper_1802_05065_b200 import units

DEVICE = dict(R=250.0, C=88e-15, I0=0.748e-6, T=1.2)


def test_device_of_the_paper():
    n = ou.paper_normalisation(**DEVICE)
    ramp = 1.0 / 200.0                                      # 200 Hz sweep
    steps = ramp / n["time_unit"] / 1e-4                    # h = 1e-4 in the paper's time unit
    assert 1.0 / steps == pytest.approx(1.8e-12, rel=0.05)  # "about 1e-12" per step
    period = 2.0 * math.pi / math.sqrt(n["V0"])             # plasma period in the paper's time unit
    assert 1e-4 / period == pytest.approx(2.3e-4, rel=0.05) # "about 2e-4" of a period
    lib = ou.library_parameters(**DEVICE, ramp_time=ramp)
    assert n["V0"] == pytest.approx(211.0, rel=0.01) and lib["omega_p"] == pytest.approx(1.61e11, rel=0.01)
    assert lib["alpha"] == pytest.approx(0.283, rel=0.01) and lib["temperature"] == pytest.approx(0.0673, rel=0.01)
    assert lib["nu"] == pytest.approx(1.24e-9, rel=0.01)


def test_front_end_agrees_with_the_paper_route():
    for dev in (DEVICE, dict(R=50.0, C=1e-12, I0=10e-6, T=4.2), dict(R=1e3, C=5e-15, I0=0.1e-6, T=0.05)):
        want = ou.library_parameters(**dev, ramp_time=2e-3)
        got = units.junction_params(dev["R"], dev["C"], dev["I0"], dev["T"], ramp_time_s=2e-3)
        for k in ("alpha", "temperature", "nu", "omega_p"):
            assert got[k] == pytest.approx(want[k], rel=1e-12), k
        n = ou.paper_normalisation(**dev)
        assert got["beta"] == pytest.approx(n["beta"], rel=1e-12) and got["v0"] == pytest.approx(n["V0"], rel=1e-12)
        # fluctuation-dissipation survives the rescaling: D / V0^(3/2) = alpha * T
        assert got["alpha"] * got["temperature"] == pytest.approx(n["D"] / n["V0"] ** 1.5, rel=1e-12)
    assert units.junction_params(250.0, 88e-15, 0.748e-6, 1.2)["nu"] == 0.0
    with pytest.raises(ValueError):
        units.junction_params(0.0, 1e-12, 1e-6, 1.0)
