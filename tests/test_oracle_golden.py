"""Pins the oracle's codecs to the values the paper itself prints (tests/golden/paper_closed_forms.txt)."""
import os

import numpy as np

from oracle import hif4_oracle as ho
from oracle import sharq_oracle as so

HERE = os.path.dirname(os.path.abspath(__file__))


def golden():
    out = {}
    for line in open(os.path.join(HERE, "golden", "paper_closed_forms.txt")):
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split("=")
            out[k.strip()] = [float(t) for t in v.split()]
    return out


def test_nvfp4_closed_forms():
    g = golden()
    assert list(so.E2M1_VALUES) == g["e2m1_magnitudes"]
    assert list(so.e2m1_decode(np.arange(8, dtype=np.uint8))) == g["e2m1_magnitudes"]
    assert float(so.e4m3_decode(np.array([0x7E], dtype=np.uint8))[0]) == g["e4m3_max"][0]
    assert float(so.PTS_TARGET) == g["nvfp4_pts_target"][0] == g["e4m3_max"][0] * g["e2m1_magnitudes"][-1]
    assert g["nvfp4_global_max_mantissa"][0] * 2.0 ** g["nvfp4_global_max_exponent"][0] == g["nvfp4_pts_target"][0]
    # smallest positive NVFP4 magnitude = smallest E4M3 subnormal (2^-9) * smallest E2M1 step (0.5)
    assert float(so.e4m3_decode(np.array([1], dtype=np.uint8))[0]) * 0.5 == 2.0 ** g["nvfp4_min_positive_log2"][0]


def test_hif4_closed_forms():
    g = golden()
    assert g["hif4_unit_elements"][0] * 4 + 32 == g["hif4_unit_bits"][0]
    assert float(ho.e6m2_decode(np.array([int(g["e6m2_max_code"][0])], dtype=np.uint8))[0]) == g["e6m2_max_value"][0]
    assert float(ho.e6m2_decode(np.array([0], dtype=np.uint8))[0]) == 2.0 ** g["e6m2_min_log2"][0]
    # largest / smallest magnitude inside a unit relative to its E6M2 scale (Eq. 15 with both shift bits set)
    codes = np.array([[7] + [1] * 63], dtype=np.uint8)            # S1P2 1.75 and 0.25
    meta = np.array([(48 << 2) | (0xFF << 8) | (0xFFFF << 16)], dtype=np.uint32)   # E6M2 = 1.0, all E1 bits set
    v = ho.hif4_decode_units(codes, meta)[0]
    assert float(v[0]) == g["hif4_in_unit_max"][0]
    codes0 = np.array([[1] * 64], dtype=np.uint8)
    meta0 = np.array([48 << 2], dtype=np.uint32)                  # no shift
    assert float(ho.hif4_decode_units(codes0, meta0)[0, 0]) == g["hif4_in_unit_min"][0]
    gmax = g["e6m2_max_value"][0] * g["hif4_in_unit_max"][0]
    assert gmax == g["hif4_global_max_mantissa"][0] * 2.0 ** g["hif4_global_max_exponent"][0]
    assert 2.0 ** g["e6m2_min_log2"][0] * g["hif4_in_unit_min"][0] == 2.0 ** g["hif4_global_min_log2"][0]
