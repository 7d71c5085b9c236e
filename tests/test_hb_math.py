"""The heatbath's double-precision elementary functions (paper_1310_7087_b200/csrc/hb_math.cuh) evaluated on the HOST against
libm in long double: the same source the kernels compile, with the hardware seeds replaced by 20-bit host seeds.  Pins the
error bounds the header states (and through them the claim that the fp64 heatbath stays within 1e-12 of the oracle, whose
accept decisions it shares).  No GPU, no oracle."""
import os
import subprocess

import pytest

HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module")
def maxima(tmp_path_factory):
    exe = str(tmp_path_factory.mktemp("hbm") / "hb_math_host")
    # -ffp-contract=off: only the fused multiply-adds the source writes (std::fma), as on the device
    subprocess.run(["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-o", exe, os.path.join(HERE, "hb_math_host.cpp")], check=True)
    out = subprocess.run([exe], check=True, capture_output=True, text=True).stdout.split()
    return [float(x) for x in out]


def test_log_of_a_uniform(maxima):
    # |ln u| <= 33 ln 2 = 22.9: 5e-15 absolute is ~1.4 units in the last place of the largest results
    assert maxima[0] < 5e-15


def test_cos_squared_sin_cos(maxima):
    assert maxima[1] < 4e-16 and maxima[2] < 4e-16 and maxima[3] < 4e-16


def test_sqrt_rsqrt_rcp(maxima):
    assert maxima[4] < 3e-16 and maxima[5] < 3e-16 and maxima[6] < 3e-16
    assert maxima[7] == 0.0 and maxima[8] == 0.0          # sqrt_pos(0) = 0, radicands below 1e-300 flush to 0
