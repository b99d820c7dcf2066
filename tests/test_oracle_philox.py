"""Pins P1, P2: the oracle's noise generator against published known-answer
vectors, the exact uniform lattice, and the moments of the normals (eq.(3))."""
import numpy as np

from oracle import oracle as O


def _read_kat(path):
    rows = []
    for line in path.read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        w = [int(t, 16) for t in line.split()]
        rows.append((w[0:4], w[4:6], w[6:10]))
    return rows


def test_philox_known_answers(golden_dir):
    rows = _read_kat(golden_dir / "philox_kat.txt")
    assert len(rows) == 3
    for ctr, key, out in rows:
        assert O.philox4x32_10(ctr, key) == out


def test_philox_counter_word_order_matters():
    # a transposed counter or key word must change the stream
    a = O.philox4x32_10([1, 2, 3, 4], [5, 6])
    assert a != O.philox4x32_10([2, 1, 3, 4], [5, 6])
    assert a != O.philox4x32_10([1, 2, 4, 3], [5, 6])
    assert a != O.philox4x32_10([1, 2, 3, 4], [6, 5])


def test_uniform_lattice_is_exact_and_open():
    # [R-2]: u = (2 (r>>9) + 1) 2^-24 is a 24-bit odd integer over 2^24: exact in fp32 and fp64
    for r in (0, 1, 511, 512, 0x7FFFFFFF, 0x80000000, 0xFFFFFFFF, 0x6627E8D5):
        u = O.uniform(r)
        assert 0.0 < u < 1.0
        assert float(np.float32(u)) == u
        assert u * 2 ** 24 == 2 * (r >> 9) + 1
    assert O.uniform(0) == 2.0 ** -24
    assert O.uniform(0xFFFFFFFF) == 1.0 - 2.0 ** -24


def test_normals_worked_example(golden_dir):
    vals = {}
    for line in (golden_dir / "worked_example_cfg0.txt").read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        vals[k] = np.array([float(t) for t in v])
    r = O.philox4x32_10([0, 0, 0, 0], [0, 0])
    np.testing.assert_allclose([O.uniform(w) for w in r], vals["uniforms"], atol=6e-10)
    for key, (k, t, it, b) in {"z_k0_t0_i0_b0": (0, 0, 0, 0), "z_k1_t0_i0_b0": (1, 0, 0, 0),
                               "z_k0_t1_i0_b0": (0, 1, 0, 0), "z_k255_t19_i0_b0": (255, 19, 0, 0),
                               "z_k4095_t49_i9_b0": (4095, 49, 9, 0)}.items():
        np.testing.assert_allclose(O.normals(0, k, t, it, b), vals[key], atol=2e-12, rtol=0)


def test_normals_seed_goes_in_the_key():
    z = O.normals(0x0000000100000002, 3, 4, 5, 6)
    r = O.philox4x32_10([3, 4, 5, 6], [2, 1])
    rad = np.sqrt(-2 * np.log(O.uniform(r[0])))
    assert abs(z[0] - rad * np.cos(2 * np.pi * O.uniform(r[1]))) < 1e-14
    assert abs(z[1] - rad * np.sin(2 * np.pi * O.uniform(r[1]))) < 1e-14


def test_normal_moments():
    # P2: 2.5e5 (k,t) blocks -> 1e6 draws; N(0,1) to sampling accuracy
    z = np.array([O.normals(7, k, t, 1, 0) for k in range(5000) for t in range(50)]).ravel()
    n = z.size
    assert abs(z.mean()) < 4.0 / np.sqrt(n)
    assert abs(z.var() - 1.0) < 5e-3
    assert abs(np.mean(z ** 4) / z.var() ** 2 - 3.0) < 2e-2
    # the four rotor streams are uncorrelated
    zz = z.reshape(-1, 4)
    c = np.corrcoef(zz.T) - np.eye(4)
    assert np.abs(c).max() < 6e-3
