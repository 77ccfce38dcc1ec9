"""Pins for the seeded input generators (no GPU)."""
import os

import numpy as np

from paper_1410_6685_b200 import inputs

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def test_splitmix64_published_vectors():
    want = [int(l, 16) for l in open(os.path.join(GOLDEN, "splitmix64_vectors.txt")) if l.startswith("0x")]
    got = [inputs._mix_int((i + 1) * 0x9E3779B97F4A7C15) for i in range(3)]
    assert got == want


def test_vector_form_equals_scalar_form_and_is_chunk_independent():
    for seed, stream in [(1, 0), (3, 2), (5, 0)]:
        v = inputs.bits(seed, stream, 1000, 50)
        assert v.tolist() == [inputs.bits_scalar(seed, stream, 1000 + i) for i in range(50)]
    a = inputs.uniform_pm1_f64(1, 0, inputs._CHUNK + 17)
    assert a[inputs._CHUNK + 3] == 2.0 * (inputs.bits_scalar(1, 0, inputs._CHUNK + 3) >> 11) * 2.0 ** -53 - 1.0
    assert (a >= -1).all() and (a < 1).all() and abs(a.mean()) < 1e-2


def test_distributions():
    x = inputs.normal_f32(2, 0, 1 << 18)
    assert x.dtype == np.float32 and abs(x.mean()) < 1e-2 and abs(x.std() - 1) < 1e-2 and np.isfinite(x).all()
    i = inputs.uniform_i31(3, 0, 1 << 18)
    assert i.dtype == np.int32 and i.min() >= 0 and abs(np.mean(i % 7 == 3) - 1 / 7) < 5e-3
    s = inputs.sorted_cumsum_f32(4, 0, inputs._CHUNK + 100)
    assert (np.diff(s) >= 0).all() and s[0] >= 0
    u = inputs.u01(4, 0, 0, inputs._CHUNK + 100)
    assert s[-1] == np.float32(np.cumsum(u)[-1])          # chunk carry keeps the sequential order
    m = inputs.boosted_matrix_f64(5, 0, 64)
    assert (np.abs(np.diag(m) - 64) <= 1).all() and (np.abs(m - np.diag(np.diag(m))) < 1).all()
    assert inputs.checksum(m) == inputs.checksum(m.copy()) != inputs.checksum(m + 1)
