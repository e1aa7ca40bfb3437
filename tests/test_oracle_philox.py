"""Pins of the oracle's Philox sampler (reading P4): Random123 KAT, cuRAND host generator, ranges."""
import ctypes
import os

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")


def test_philox_kat(orc):
    rows = [l.split() for l in open(GOLD) if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for row in rows:
        v = [int(x, 16) for x in row]
        out = orc.philox4x32_10(v[0:4], v[4:6])
        assert [int(x) for x in out] == v[6:10]


def _curand_host(seed, offset, n):
    try:
        lib = ctypes.CDLL("libcurand.so")
    except OSError:
        try:
            lib = ctypes.CDLL("/usr/local/cuda/lib64/libcurand.so")
        except OSError:
            pytest.skip("libcurand not found")
    gen = ctypes.c_void_p()
    if lib.curandCreateGeneratorHost(ctypes.byref(gen), 161) != 0:  # CURAND_RNG_PHILOX4_32_10
        pytest.skip("cuRAND host generator unavailable")
    assert lib.curandSetPseudoRandomGeneratorSeed(gen, ctypes.c_ulonglong(seed)) == 0
    assert lib.curandSetGeneratorOffset(gen, ctypes.c_ulonglong(offset)) == 0
    out = np.zeros(n, dtype=np.uint32)
    assert lib.curandGenerate(gen, out.ctypes.data_as(ctypes.c_void_p), ctypes.c_size_t(n)) == 0
    lib.curandDestroyGenerator(gen)
    return out


@pytest.mark.parametrize("seed", [0, 1, 0x299F31D0A4093822, 0xFFFFFFFFFFFFFFFF])
def test_philox_matches_curand_host(orc, seed):
    """cuRAND host default ordering: output block i = counter (0, 0, i, 0) (subsequence i) under
    key (seed_lo, seed_hi).  Pins the c2 lane and both key words."""
    n_blocks = 64
    ref = _curand_host(seed, 0, 4 * n_blocks)
    key = [seed & 0xFFFFFFFF, seed >> 32]
    got = np.concatenate([orc.philox4x32_10([0, 0, i, 0], key) for i in range(n_blocks)])
    np.testing.assert_array_equal(got, ref)


def test_philox_counter_high_word_vs_curand_offset(orc):
    """The host stream interleaves 65536 subsequences of 4 words, so offset 4*65536*(2^32+5) lands
    on counter (5, 1, i, 0): pins the c0 and c1 lanes."""
    seed = 12345
    ref = _curand_host(seed, 4 * 65536 * ((1 << 32) + 5), 8)
    key = [seed & 0xFFFFFFFF, seed >> 32]
    got = np.concatenate([orc.philox4x32_10([5, 1, 0, 0], key), orc.philox4x32_10([5, 1, 1, 0], key)])
    np.testing.assert_array_equal(got, ref)


def test_uniform_map(orc):
    assert orc.uniform_f32(0, 2.0, 5.0) == 2.0
    top = orc.uniform_f32(0xFFFFFFFF, 0.0, 1.0)
    assert top == 1.0 - 2.0 ** -24
    assert orc.uniform_f32(0x80000000, -1.0, 1.0) == 0.0
    # low 8 bits are dropped
    assert orc.uniform_f32(0x12345600, 0.0, 1.0) == orc.uniform_f32(0x123456FF, 0.0, 1.0)
    # one fp32 fma: compare with exact rational arithmetic rounded once
    w, lo, hi = 0xDEADBEEF, np.float32(-3.3), np.float32(7.7)
    span = np.float32(hi - lo)
    exact = (w >> 8) * 2.0 ** -24 * float(span) + float(lo)
    assert orc.uniform_f32(w, float(lo), float(hi)) == float(np.float32(exact))


def test_draw_word_keying(orc):
    """Every key component (seed, it, r, s, kind, k, block) changes the stream; word j&3 of block j>>2."""
    base = dict(seed=7, it=3, r=2, s=11, kind=1, k=5, j=0)
    w0 = orc.draw_word(**base)
    for name, val in [("seed", 8), ("it", 4), ("r", 3), ("s", 12), ("kind", 0), ("k", 6), ("j", 4)]:
        assert orc.draw_word(**{**base, name: val}) != w0
    key = [7, 0]
    for j in range(12):
        blk = orc.philox4x32_10([3, 2, 11, (1 << 31) | (5 << 4) | (j >> 2)], key)
        assert orc.draw_word(**{**base, "j": j}) == int(blk[j & 3])


def test_samplers_in_bounds_and_uniform(orc):
    from paper_2607_03987_b200 import workloads as wl
    for name in ("C1", "C3", "C4"):
        p, _ = wl.CONFIGS[name]()
        op = orc.OracleProblem(p)
        xs = np.array([op.sample_state(5, 1, 2, s) for s in range(2000)])
        us = np.array([op.sample_control(5, 1, 2, s, s % 7) for s in range(2000)])
        for d in range(p.state_dim):
            if p.dim_kind[d] == wl.DIM_ANGLE:
                assert np.all(xs[:, d] >= -np.float32(np.pi)) and np.all(xs[:, d] < np.float32(np.pi))
            else:
                assert np.all(xs[:, d] >= p.state_lo[d]) and np.all(xs[:, d] <= p.state_hi[d])
                mid = 0.5 * (p.state_lo[d] + p.state_hi[d])
                span = p.state_hi[d] - p.state_lo[d]
                assert abs(xs[:, d].mean() - mid) < 0.05 * span  # ~2.7 sigma at n=2000 is 0.017*span
        assert np.all(us >= p.control_lo) and np.all(us <= p.control_hi)
        # values are fp32-representable (P4: sample evaluated in fp32 on both sides)
        assert np.array_equal(xs, xs.astype(np.float32).astype(np.float64))
        # chi-square smoke test on the first state dim, 16 bins
        h, _ = np.histogram(xs[:, 0], bins=16, range=(p.state_lo[0], p.state_hi[0]))
        chi2 = ((h - 125.0) ** 2 / 125.0).sum()
        assert chi2 < 45.0  # 15 dof, p ~ 1e-4
