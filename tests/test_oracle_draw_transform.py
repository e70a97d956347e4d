"""Pins for the oracle's draw (o1) and sampled transform (o2-o4).  CPU only.

Every check compares the C oracle with something that is not the oracle: the published
splitmix64 vector, a pure-Python big-int restatement of the draw rule, the defining cosine sum
written out here, closed forms, numpy.fft (test-only cross-check).
"""
import os

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden")
MASK = (1 << 64) - 1


def py_splitmix(seed, k):
    z = (seed + (k + 1) * 0x9E3779B97F4A7C15) & MASK
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & MASK
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & MASK
    return z ^ (z >> 31)


def py_draw(m, s, seed):
    """DESIGN.md reading R1, restated with Python integers."""
    nw = (m + 63) // 64
    signs = [py_splitmix(seed, w) for w in range(nw)]
    B = m // 2 + 1
    kept, k = [], nw
    while len(kept) < s:
        c = (py_splitmix(seed, k) * B) >> 64
        if c not in kept:
            kept.append(c)
        k += 1
    return signs, sorted(kept), k


def test_splitmix64_published_vector(orc):
    want = [int(l) for l in open(os.path.join(GOLD, "splitmix64_seed1234567.txt")) if not l.startswith("#")]
    got = [orc.splitmix64_at(1234567, k) for k in range(len(want))]
    assert got == want


def test_splitmix64_counter_form_matches_sequential_state(orc):
    # sequential reference generator: state += gamma; return mix(state)
    state = 42
    for k in range(50):
        state = (state + 0x9E3779B97F4A7C15) & MASK
        z = state
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & MASK
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & MASK
        assert orc.splitmix64_at(42, k) == (z ^ (z >> 31))


@pytest.mark.parametrize("m,s,seed", [(4096, 32, 2), (64, 33, 7), (100, 10, 3), (1 << 14, 512, 99), (2, 2, 0)])
def test_draw_matches_python_restatement(orc, m, s, seed):
    signs, idx = orc.draw(m, s, seed)
    psigns, pidx, _ = py_draw(m, s, seed)
    assert [int(x) for x in signs] == psigns
    assert [int(x) for x in idx] == pidx
    assert len(set(pidx)) == s and min(pidx) >= 0 and max(pidx) <= m // 2
    assert list(idx) == sorted(idx)


def test_draw_survey_values(orc):
    # (m=4096, s=32, seed=2) consumes stream positions 64..95
    signs, idx = orc.draw(4096, 32, 2)
    assert list(idx[:8]) == [11, 152, 248, 353, 362, 442, 471, 505]
    assert list(idx[-3:]) == [1905, 1913, 1976]
    assert [(int(signs[0]) >> t) & 1 for t in range(16)] == [0, 1, 1, 1, 0, 0, 1, 1, 0, 1, 1, 0, 1, 0, 1, 0]
    assert py_draw(4096, 32, 2)[2] == 96


def test_draw_sign_balance_and_full_range(orc):
    signs, _ = orc.draw(1 << 16, 8, 5)
    ones = sum(bin(int(w)).count("1") for w in signs)
    assert abs(ones / (1 << 16) - 0.5) < 0.01
    # s = B: every bin must appear exactly once
    _, idx = orc.draw(64, 33, 11)
    assert list(idx) == list(range(33))
    with pytest.raises(ValueError):
        orc.draw(64, 34, 11)


def dft_direct(x):
    m = len(x)
    t = np.arange(m)
    out = np.zeros(m, dtype=complex)
    for k in range(m):
        ang = -2.0 * np.pi * ((k * t) % m) / m
        out[k] = np.sum(x * (np.cos(ang) + 1j * np.sin(ang)))
    return out


@pytest.mark.parametrize("m", [1, 2, 4, 8, 64, 512])
def test_fft_vs_direct_sum(orc, m):
    rng = np.random.default_rng(m)
    x = rng.standard_normal(m) + 1j * rng.standard_normal(m)
    got = orc.fft(x)
    want = dft_direct(x)
    assert np.max(np.abs(got - want)) <= 1e-13 * max(1.0, np.linalg.norm(x)) * np.sqrt(m)


def test_fft_closed_forms(orc):
    m = 256
    t = np.arange(m)
    # impulse at t0 -> exp(-2 pi i k t0/m)
    x = np.zeros(m); x[5] = 1.0
    k = np.arange(m)
    assert np.allclose(orc.fft(x), np.exp(-2j * np.pi * k * 5 / m), atol=1e-14)
    # constant -> m at bin 0
    X = orc.fft(np.ones(m))
    assert abs(X[0] - m) < 1e-12 and np.max(np.abs(X[1:])) < 1e-12
    # pure cosine at k0 -> m/2 at k0 and m-k0
    X = orc.fft(np.cos(2 * np.pi * 7 * t / m))
    want = np.zeros(m); want[7] = want[m - 7] = m / 2
    assert np.max(np.abs(X - want)) < 1e-11
    # Nyquist cosine -> m at m/2
    X = orc.fft(np.cos(np.pi * t))
    assert abs(X[m // 2] - m) < 1e-11


def test_fft_hermitian_parseval_linearity_numpy(orc):
    m = 1024
    rng = np.random.default_rng(0)
    x, y = rng.standard_normal(m), rng.standard_normal(m)
    X, Y = orc.fft(x), orc.fft(y)
    # Hermitian symmetry of a real input
    assert np.max(np.abs(X[1:][::-1] - np.conj(X[1:]))) < 1e-11
    # Parseval
    assert abs(np.sum(np.abs(X) ** 2) - m * np.sum(x ** 2)) < 1e-9 * m * np.sum(x ** 2)
    # linearity
    assert np.max(np.abs(orc.fft(2 * x - 3 * y) - (2 * X - 3 * Y))) < 1e-10
    # test-only cross-check with numpy's FFT (sign convention e^{-i...})
    assert np.max(np.abs(X - np.fft.fft(x))) < 1e-11


def sketch_brute(A, signs, idx):
    """sqrt(s/m) * sum_t d_t a_t cos(2 pi k_i t/m), the definition (north_star: O(m s) direct sum)."""
    m, n = A.shape
    s = len(idx)
    d = np.array([-1.0 if (int(signs[t >> 6]) >> (t & 63)) & 1 else 1.0 for t in range(m)])
    t = np.arange(m)
    out = np.zeros((s, n))
    for i, k in enumerate(idx):
        c = np.cos(2.0 * np.pi * ((int(k) * t) % m) / m)
        for j in range(n):
            out[i, j] = np.sqrt(s / m) * float(np.sum(np.longdouble(d * A[:, j]) * np.longdouble(c)))
    return out


@pytest.mark.parametrize("m,n,s", [(4096, 5, 12), (256, 3, 129), (1000, 4, 9), (96, 2, 5)])
def test_sketch_vs_bruteforce(orc, m, n, s):
    rng = np.random.default_rng(m + n)
    A = np.asfortranarray(rng.standard_normal((m, n)))
    signs, idx = orc.draw(m, s, 17)
    got = orc.sketch(A, signs, idx)
    want = sketch_brute(A, signs, idx)
    assert np.linalg.norm(got - want) <= 1e-13 * np.linalg.norm(want) * np.sqrt(m)


def test_sketch_impulse_and_sign_flip(orc):
    m, s = 512, 16
    signs, idx = orc.draw(m, s, 3)
    d = np.array([-1.0 if (int(signs[t >> 6]) >> (t & 63)) & 1 else 1.0 for t in range(m)])
    A = np.zeros((m, 2), order="F")
    A[37, 0] = 1.0
    A[:, 1] = d            # D*A[:,1] = ones -> only bin 0 is non-zero
    As = orc.sketch(A, signs, idx)
    want0 = np.sqrt(s / m) * d[37] * np.cos(2 * np.pi * idx * 37 / m)
    assert np.max(np.abs(As[:, 0] - want0)) < 1e-14
    want1 = np.where(idx == 0, np.sqrt(s / m) * m, 0.0)
    assert np.max(np.abs(As[:, 1] - want1)) < 1e-11


# ---- Re+Im variant of the sketch -------------------------------------------------
def sketch_im_brute(A, signs, idx):
    """sqrt(s/m) * Im sum_t d_t a_t exp(-2 pi i k_i t/m) = -sqrt(s/m) sum_t d_t a_t sin(2 pi k_i t/m)."""
    m, n = A.shape
    s = len(idx)
    d = np.array([-1.0 if (int(signs[t >> 6]) >> (t & 63)) & 1 else 1.0 for t in range(m)])
    t = np.arange(m)
    out = np.zeros((s, n))
    for i, k in enumerate(idx):
        sn = np.sin(2.0 * np.pi * ((int(k) * t) % m) / m)
        for j in range(n):
            out[i, j] = -np.sqrt(s / m) * float(np.sum(np.longdouble(d * A[:, j]) * np.longdouble(sn)))
    return out


@pytest.mark.parametrize("m,n,s", [(4096, 5, 12), (256, 3, 129), (1000, 4, 9), (96, 2, 5)])
def test_sketch_reim_vs_bruteforce(orc, m, n, s):
    rng = np.random.default_rng(3 * m + n)
    A = np.asfortranarray(rng.standard_normal((m, n)))
    signs, idx = orc.draw(m, s, 19)
    got = orc.sketch_reim(A, signs, idx)
    assert got.shape == (2 * s, n)
    # the Re rows are the Re-only sketch, bit for bit (same transform, same gather, same scale)
    assert np.array_equal(got[:s], orc.sketch(A, signs, idx)) or m & (m - 1)
    want_re, want_im = sketch_brute(A, signs, idx), sketch_im_brute(A, signs, idx)
    tol = 1e-13 * np.sqrt(m)
    assert np.linalg.norm(got[:s] - want_re) <= tol * np.linalg.norm(want_re)
    assert np.linalg.norm(got[s:] - want_im) <= tol * max(np.linalg.norm(want_im), np.linalg.norm(want_re))


def test_sketch_reim_closed_forms(orc):
    """Column j = d * sin(2 pi k_j t/m): X[k_j] = -i m/2, so Im = -m/2 at (s + j, j) and nothing else (bins are
    distinct and below m/2 or at 0 / m/2); a constant column d * 1 has Im = 0 everywhere; Im X[0] = Im X[m/2] = 0."""
    m, n, s = 1024, 6, 24
    signs, idx = orc.draw(m, s, 11)
    d = np.array([-1.0 if (int(signs[t >> 6]) >> (t & 63)) & 1 else 1.0 for t in range(m)])
    t = np.arange(m)
    cols, live = [], []
    for j in range(n - 1):
        k0 = int(idx[j])
        cols.append(d * np.sin(2 * np.pi * k0 * t / m))
        live.append(k0 not in (0, m // 2))
    cols.append(d.copy())
    A = np.asfortranarray(np.stack(cols, axis=1))
    As = orc.sketch_reim(A, signs, idx)
    scale = np.sqrt(s / m)
    want = np.zeros((2 * s, n))
    for j in range(n - 1):
        if live[j]:
            want[s + j, j] = -0.5 * m * scale
    want[:s, n - 1] = np.where(idx == 0, m * scale, 0.0)
    assert np.max(np.abs(As - want)) < 1e-10
    # a generic real column: the imaginary part vanishes at DC and Nyquist
    rng = np.random.default_rng(5)
    B = np.asfortranarray(rng.standard_normal((m, 1)))
    idx2 = np.array([0, m // 2, 3], dtype=np.int64)
    As2 = orc.sketch_reim(B, signs, idx2)
    assert abs(As2[3, 0]) < 1e-12 and abs(As2[4, 0]) < 1e-12 and abs(As2[5, 0]) > 1e-6
