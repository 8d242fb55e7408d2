"""Pins for the oracle's primitives (R1-R4, R8): each test checks the oracle against something
other than itself -- published vectors, an independent library, exact rational arithmetic,
mpmath -- so that a wrong constant, sign, index or operand order fails here."""
import ctypes
import os
from fractions import Fraction

import mpmath as mp
import numpy as np
import pytest

import oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(path, tag=None):
    out = []
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        parts = line.split()
        if tag is None:
            out.append(parts)
        elif parts[0] == tag:
            out.append(parts[1:])
    return out


# ---------------------------------------------------------------- R1 Philox
def test_philox_published_kat():
    rows = _rows(os.path.join(GOLD, "philox4x32_10_kat.txt"))
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        assert list(O.philox4x32_10(v[0:4], v[4:6])) == v[6:10]


def _py_philox(c, k):
    """Second, independent restatement (Python big ints) used to check the C++ on random inputs."""
    c = list(c)
    k = list(k)
    for _ in range(10):
        p0 = 0xD2511F53 * c[0]
        p1 = 0xCD9E8D57 * c[2]
        c = [(p1 >> 32) ^ c[1] ^ k[0], p1 & 0xFFFFFFFF, (p0 >> 32) ^ c[3] ^ k[1], p0 & 0xFFFFFFFF]
        k = [(k[0] + 0x9E3779B9) & 0xFFFFFFFF, (k[1] + 0xBB67AE85) & 0xFFFFFFFF]
    return c


def test_philox_vs_python_bigint_random():
    rng = np.random.default_rng(0)
    for _ in range(200):
        c = [int(x) for x in rng.integers(0, 2**32, 4)]
        k = [int(x) for x in rng.integers(0, 2**32, 2)]
        assert [int(x) for x in O.philox4x32_10(c, k)] == _py_philox(c, k)


def _curand_host(seed, n, offset=0):
    path = "/usr/local/cuda/lib64/libcurand.so"
    if not os.path.exists(path):
        pytest.skip("libcurand not present")
    cr = ctypes.CDLL(path)
    gen = ctypes.c_void_p()
    if cr.curandCreateGeneratorHost(ctypes.byref(gen), 161) != 0:  # CURAND_RNG_PHILOX4_32_10
        pytest.skip("cuRAND host generator unavailable")
    assert cr.curandSetPseudoRandomGeneratorSeed(gen, ctypes.c_ulonglong(seed)) == 0
    assert cr.curandSetGeneratorOffset(gen, ctypes.c_ulonglong(offset)) == 0
    out = (ctypes.c_uint * n)()
    assert cr.curandGenerate(gen, out, n) == 0
    cr.curandDestroyGenerator(gen)
    return list(out)


def test_philox_vs_curand_host_library():
    """cuRAND's host Philox4x32-10: the first 4 outputs are Philox(ctr=(0,0,0,0), key=(seed_lo, seed_hi)),
    the next 4 come from subsequence 1, i.e. ctr=(0,0,1,0). An independent library implementation."""
    for seed in (0, 1, 0x0000000600000005, 0xDEADBEEFCAFEF00D):
        key = [seed & 0xFFFFFFFF, seed >> 32]
        got = _curand_host(seed, 16)
        for sub in range(4):
            assert [int(x) for x in O.philox4x32_10([0, 0, sub, 0], key)] == got[4 * sub:4 * sub + 4]


# ---------------------------------------------------------------- R3 stream layout
def test_derived_keys_and_words_match_worked_example():
    f = os.path.join(GOLD, "config1_worked.txt")
    for r in _rows(f, "derived_key"):
        seed = int(r[0].split("=")[1])
        assert [f"{x:08x}" for x in O.derive_key(seed, 0)] == r[1:3]
    (r,) = _rows(f, "philox")
    v = [int(x, 16) for x in r]
    assert list(O.philox4x32_10(v[0:4], v[4:6])) == v[6:10]
    (words,) = _rows(f, "words")
    assert [f"{x:08x}" for x in O.unit_words(1, 0, 0, 1, 0, 0, 12)] == words


def test_stream_layout_counter_fields():
    """Word idx lives in call q = idx>>2, lane idx&3, counter (q, t | l<<8 | P[79:64]<<16, P[31:0], P[63:32])."""
    seed, inst = 0x1234567890ABCDEF, 7
    key = O.derive_key(seed, inst)
    # derived key definition
    assert list(key) == list(O.philox4x32_10([inst, 0, 0, 0x5A4D4321], [seed & 0xFFFFFFFF, seed >> 32])[:2])
    P = (0xBEEF << 64) | (0x89ABCDEF << 32) | 0x01234567
    level, trial = 5, 200
    first, n = 4 * 1000 + 3, 10
    got = O.unit_words(seed, inst, P, level, trial, first, n)
    exp = []
    for idx in range(first, first + n):
        q = idx >> 2
        out = _py_philox([q, trial | (level << 8) | (0xBEEF << 16), 0x01234567, 0x89ABCDEF], [int(key[0]), int(key[1])])
        exp.append(out[idx & 3])
    assert [int(x) for x in got] == exp
    # distinct units give distinct streams
    a = O.unit_words(seed, inst, P, level, trial, 0, 8)
    for other in (O.unit_words(seed, inst, P + 1, level, trial, 0, 8), O.unit_words(seed, inst, P, level + 1, trial, 0, 8),
                  O.unit_words(seed, inst, P, level, trial + 1, 0, 8), O.unit_words(seed, inst + 1, P, level, trial, 0, 8),
                  O.unit_words(seed + 1, inst, P, level, trial, 0, 8), O.unit_words(seed, inst, P ^ (1 << 70), level, trial, 0, 8)):
        assert list(a) != list(other)


# ---------------------------------------------------------------- R2 geometry
def test_geometry_exact_rational():
    lower, upper, g, level = [0.0, -1.0, 2.5], [10.0, 1.0, 7.0], 3, 3
    coords = [26, 0, 13]
    lo, w, V = O.cell_geometry(3, lower, upper, g, level, coords)
    for d in range(3):
        we = (Fraction(upper[d]) - Fraction(lower[d])) / g**level
        assert abs(Fraction(w[d]) - we) <= abs(we) * Fraction(1, 2**52)
        assert abs(Fraction(lo[d]) - (Fraction(lower[d]) + coords[d] * we)) <= Fraction(1, 2**49)
    assert V == w[0] * w[1] * w[2]


def test_children_tile_parent():
    """Children of a cell: union of boxes = parent box (integer coordinates), volumes add up."""
    dim, g = 3, 4
    lower, upper = [0.0] * 3, [10.0] * 3
    P, pc = O.path_coords(dim, g, [37])
    plo, pw, pV = O.cell_geometry(dim, lower, upper, g, 1, pc)
    seen = set()
    vol = 0.0
    for j in range(g**dim):
        Pc, cc = O.path_coords(dim, g, [37, j])
        assert Pc == P * g**dim + j
        for d in range(dim):
            assert cc[d] // g == pc[d]
        seen.add(tuple(c % g for c in cc))
        lo, w, V = O.cell_geometry(dim, lower, upper, g, 2, cc)
        vol += V
        for d in range(dim):
            assert lo[d] >= plo[d] - 1e-15 and lo[d] + w[d] <= plo[d] + pw[d] + 1e-14
    assert len(seen) == g**dim
    assert abs(vol - pV) <= 1e-15 * pV * g**dim
    # axis 0 is the least significant digit of j
    assert O.path_coords(dim, g, [1])[1] == [1, 0, 0] and O.path_coords(dim, g, [g])[1] == [0, 1, 0]


# ---------------------------------------------------------------- R4 map
def test_map_f64_lattice():
    lo, w = 2.5, 1.25
    assert O.map_f64(0, lo, w) == lo + 0.5 * w * 2.0**-32
    assert O.map_f64(2**32 - 1, lo, w) == lo + (2.0**32 - 0.5) * (w * 2.0**-32)
    assert O.map_f64(2**31, lo, w) == lo + (2.0**31 + 0.5) * (w * 2.0**-32)
    assert lo < O.map_f64(0, lo, w) and O.map_f64(2**32 - 1, lo, w) < lo + w
    f = os.path.join(GOLD, "config1_worked.txt")
    (words,) = _rows(f, "words")
    (pt,) = _rows(f, "point0")
    for d in range(3):
        assert O.map_f64(int(words[d], 16), 0.0, 2.5) == float(pt[d])


def test_map_f32_lattice_exact():
    f = os.path.join(GOLD, "config1_worked.txt")
    (words,) = _rows(f, "f32_words")
    (xb,) = _rows(f, "f32_x")
    for wd, x in zip(words, xb):
        assert f"{int(np.float32(O.map_f32(int(wd, 16), 0.0, 2.5)).view(np.uint32)):08x}" == x
    # exact rational emulation of fmaf(u', (float)w, base) with one rounding
    rng = np.random.default_rng(1)
    for _ in range(300):
        word = int(rng.integers(0, 2**32))
        lo, width, c = float(rng.uniform(-3, 3)), float(rng.uniform(0.01, 4)), float(rng.uniform(-1, 1))
        u = Fraction(1) + Fraction(word >> 9, 2**23)
        base = np.float32(np.float64((lo - width) + width * 2.0**-24) - c)
        exact = u * Fraction(float(np.float32(width))) + Fraction(float(base))
        got = O.map_f32(word, lo, width, c)
        # correctly rounded: |got - exact| <= half an ulp
        assert abs(Fraction(float(got)) - exact) <= Fraction(float(np.spacing(np.float32(abs(float(exact)))))) / 2
    # extreme words: inside the cell; the top lattice point may round onto the upper face in FP32
    assert 0.0 < float(O.map_f32(0, 0.0, 2.5)) and float(O.map_f32(2**32 - 1, 0.0, 2.5)) <= 2.5


def test_map_mean_is_cell_centre():
    words = O.unit_words(9, 0, 0, 1, 0, 0, 40000)
    x64 = np.array([O.map_f64(int(w), 1.0, 3.0) for w in words[:20000]])
    x32 = np.array([float(O.map_f32(int(w), 1.0, 3.0)) for w in words[:20000]])
    for x in (x64, x32):
        assert x.min() > 1.0 and x.max() <= 4.0
        assert abs(x.mean() - 2.5) < 4 * 3.0 / np.sqrt(12 * len(x))
        assert abs(x.var() - 9.0 / 12) < 0.03


# ---------------------------------------------------------------- R8 zsin / zexp
def test_zsin_accuracy_and_symmetry():
    mp.mp.dps = 30
    rng = np.random.default_rng(2)
    a = np.concatenate([rng.uniform(-64, 64, 4000), rng.uniform(-1e-3, 1e-3, 200), np.linspace(0, 60, 997),
                        np.array([k * np.pi for k in range(-20, 21)]), np.array([(k + 0.5) * np.pi for k in range(-20, 20)])])
    worst = 0.0
    for v in a.astype(np.float32):
        got = float(O.zsin(v))
        ref = float(mp.sin(mp.mpf(float(v))))
        worst = max(worst, abs(got - ref))
        assert float(O.zsin(-v)) == -got            # odd
    assert worst < 2.5e-7, worst                    # ~2 ulp of 1.0 (abs), argument exact in FP32
    assert float(O.zsin(np.float32(0.0))) == 0.0
    # survey pin: sum bits 4114cf10 -> sin = 0.12390633086739562 (double); zsin within 1e-7 abs
    a0 = np.array([0x4114CF10], dtype=np.uint32).view(np.float32)[0]
    assert abs(float(O.zsin(a0)) - 0.12390633086739562) < 1e-7


def test_zsin_moderate_range_degrades_gracefully():
    mp.mp.dps = 30
    rng = np.random.default_rng(3)
    for v in rng.uniform(-8000, 8000, 500).astype(np.float32):
        assert abs(float(O.zsin(v)) - float(mp.sin(mp.mpf(float(v))))) < 2e-6


def test_zexp_accuracy_and_range():
    mp.mp.dps = 30
    rng = np.random.default_rng(4)
    e = np.concatenate([rng.uniform(-700, 0, 3000), rng.uniform(-1, 1, 500), rng.uniform(0, 700, 300),
                        np.array([0.0, -0.34657, 0.34657, -87.0, -103.0, -104.0, -707.9])]).astype(np.float32)
    for v in e:
        got = O.zexp_value(v)
        ref = mp.exp(mp.mpf(float(v)))
        assert abs(mp.mpf(got) - ref) / ref < 2.5e-7, (v, got)
        p, n = O.zexp(v)
        assert 0.70 < float(p) < 1.42
    assert O.zexp_value(np.float32(0.0)) == 1.0
    assert O.zexp_value(np.float32(-709.0)) == 0.0
    assert O.zexp_value(np.float32(-1e30)) == 0.0
    assert O.zexp_value(np.float32(709.0)) == float("inf")
    assert np.isnan(O.zexp_value(np.float32("nan")))
    # well below the FP32 range the value is still resolved (reading R9)
    v = O.zexp_value(np.float32(-171.0))
    assert 0 < v < 1e-70 and abs(v / float(mp.exp(-171)) - 1) < 2.5e-7


def test_zexp_significand_and_exponent():
    for v in np.float32([-0.2, -1.0, -20.5, -171.0, 3.3]):
        p, n = O.zexp(v)
        assert n == int(np.rint(float(v) / np.log(2)))
        assert abs(float(p) - np.exp(float(v) - n * np.log(2))) < 3e-7
