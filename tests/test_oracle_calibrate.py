"""Pins for oracle O2 (calibrate) -- DESIGN.md reading S7.  CPU only."""
import numpy as np

import oracle
from bruteforce import calibrate as np_calibrate
from helpers import P


def test_all_adc_values_against_numpy_float32_steps():
    rng = np.random.default_rng(7)
    pairs = [(3.0, 20.0), (2.71828, 17.3), (3.3, 25.9), (0.0, 20.0), (1e9, 0.0), (-3.0, 20.0), (3.0, 300.0)]
    pairs += [(float(np.float32(g)), float(np.float32(p))) for g, p in zip(rng.normal(3, 0.1, 40), rng.normal(20, 2, 40))]
    for g, p in pairs:
        for adc in range(256):
            assert oracle.calibrate(adc, g, p, P) == np_calibrate(adc, g, p, P), (adc, g, p)


def test_hand_values_and_special_cases():
    # nominal: (60 - 20) * 3 * 47 - 60 = 5580 (all exactly representable)
    assert oracle.calibrate(60, 3.0, 20.0, P) == 5580
    # threshold 1000 e <=> adc <= 27 at nominal gain: (27-20)*141-60 = 927 < 1000 <= (28-20)*141-60 = 1068
    assert oracle.calibrate(27, 3.0, 20.0, P) == 927 and oracle.calibrate(28, 3.0, 20.0, P) == 1068
    assert oracle.calibrate(10, 3.0, 20.0, P) == 0             # negative -> 0
    assert oracle.calibrate(200, 0.0, 20.0, P) == 0            # masked column: 0*47 - 60 < 0
    assert oracle.calibrate(200, float("nan"), 20.0, P) == 0   # NaN -> 0
    assert oracle.calibrate(255, 1e9, 0.0, P) == 64000         # clamp
    assert oracle.calibrate(255, float("inf"), 0.0, P) == 64000
    # truncation toward zero, not rounding: f4 = (21-20)*2.5*47 - 60 = 57.5 -> 57
    assert oracle.calibrate(21, 2.5, 20.0, P) == 57
    # op order matters: ((adc-ped)*gain)*vcal, each rounded to binary32
    g, p = float(np.float32(2.9371843)), float(np.float32(19.123457))
    f = np.float32
    want = int(f(f(f(f(97) - f(p)) * f(g)) * f(47)) + f(-60))
    assert oracle.calibrate(97, g, p, P) == want
