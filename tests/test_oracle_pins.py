"""Pins for the CPU oracle: every check compares ``oracle/`` with something
that is NOT the oracle -- a closed form, a library routine, brute force, exact rationals, or an
invariant -- so that a dropped term, wrong sign, wrong index or swapped operand fails somewhere.

Definition under test (BASELINE.json:north_star):
    y_k[n] = a1_k y_k[n-1] + b0_k x[n-d_k],  y[-1]=0, x[m<0]=0;   SNR[n] = sum_k y_k[n].
"""
from fractions import Fraction
from pathlib import Path

import numpy as np
import pytest

import oracle
import spiir_inputs

GOLDEN = Path(__file__).parent / "golden"


def one_template(a1, b0, d):
    a1 = np.atleast_1d(np.asarray(a1, dtype=np.complex64))
    b0 = np.atleast_1d(np.asarray(b0, dtype=np.complex64))
    d = np.atleast_1d(np.asarray(d, dtype=np.int32))
    return np.array([0, a1.size], dtype=np.int64), a1, b0, d


def w(z):
    """float32/complex64 value widened exactly to double (what the oracle consumes)."""
    return np.asarray(z).astype(np.complex128 if np.iscomplexobj(z) else np.float64)


# ---------------------------------------------------------------- P1 impulse closed form
@pytest.mark.parametrize("d,n0", [(0, 0), (0, 5), (1, 0), (7, 3), (63, 11)])
def test_p1_impulse_closed_form(d, n0):
    N = 200
    a1 = np.complex64(0.93 * np.exp(0.37j))
    b0 = np.complex64(0.4 - 0.7j)
    x = np.zeros(N, dtype=np.float32)
    x[n0] = 1.0
    snr = oracle.run(*one_template(a1, b0, d), x)[0]
    n = np.arange(N)
    expect = np.where(n >= n0 + d, w(b0) * w(a1) ** np.maximum(n - n0 - d, 0), 0.0)
    assert np.all(snr[: n0 + d] == 0.0)                       # causal, zero pre-history
    assert np.abs(snr - expect).max() <= 1e-14 * np.abs(expect).max()


# ---------------------------------------------------------------- P2 tone closed form with transient
@pytest.mark.parametrize("r,wp,d,om", [(0.97, 0.3, 5, 0.21), (0.999, 0.02, 0, 0.02), (0.9, 1.5, 17, 0.7)])
def test_p2_tone_closed_form_with_transient(r, wp, d, om):
    N = 600
    a1 = np.complex64(r * np.exp(1j * wp))
    b0 = np.complex64(-0.3 + 0.8j)
    n = np.arange(N)
    # float32 tones are what the oracle reads; build the closed form from their exact values by
    # real-linearity: response to c[n] + i s[n], where c, s are the float32-rounded cos/sin.
    c = np.cos(om * n).astype(np.float32)
    s = np.sin(om * n).astype(np.float32)
    tpl = one_template(a1, b0, d)
    Y = oracle.run(*tpl, c)[0] + 1j * oracle.run(*tpl, s)[0]
    q = w(a1) * np.exp(-1j * om)
    m = np.maximum(n - d, 0)
    cf = np.where(n >= d, w(b0) * np.exp(1j * om * (n - d)) * (1 - q ** (m + 1)) / (1 - q), 0.0)
    # the float32 rounding of the tone (<= 6e-8 per sample) is amplified by at most |b0|/(1-|a1|)
    tol = 6e-8 * abs(w(b0)) / (1 - abs(w(a1))) * 1.5 + 1e-12
    assert np.abs(Y - cf).max() <= tol
    # late samples approach the north_star steady state b0 e^{-i om d}/(1 - a1 e^{-i om}) e^{i om n}
    if abs(q) ** (N - d) < 1e-6:
        ss = w(b0) * np.exp(-1j * om * d) / (1 - q) * np.exp(1j * om * (N - 1))
        assert abs(Y[-1] - ss) <= tol + 2 * abs(ss) * abs(q) ** (N - d)


# ---------------------------------------------------------------- P3 brute-force convolution
def test_p3_bruteforce_convolution():
    rng = np.random.default_rng(3)
    N, K = 300, 5
    a1 = (rng.uniform(0.5, 0.99, K) * np.exp(1j * rng.uniform(-3, 3, K))).astype(np.complex64)
    b0 = (rng.standard_normal(K) + 1j * rng.standard_normal(K)).astype(np.complex64)
    d = rng.integers(0, 40, K).astype(np.int32)
    x = rng.standard_normal(N).astype(np.float32)
    snr = oracle.run(*one_template(a1, b0, d), x)[0]
    A, B, X = w(a1), w(b0), w(x)
    bf = np.zeros(N, dtype=np.complex128)
    for n in range(N):
        for k in range(K):
            for j in range(0, n - int(d[k]) + 1):              # truncated impulse response
                bf[n] += B[k] * A[k] ** j * X[n - int(d[k]) - j]
    assert np.abs(snr - bf).max() <= 1e-12 * np.abs(bf).max()
    # per-filter outputs agree with the same brute force, filter by filter
    y = oracle.filter_outputs(a1, b0, d, x)
    assert np.abs(y.sum(axis=0) - snr).max() <= 1e-12 * np.abs(snr).max()


# ---------------------------------------------------------------- P4 linearity / superposition
def test_p4_linearity_union_permutation():
    inp = spiir_inputs.make_random_bank(41, [37, 64, 5], 500, d_max=100)
    rng = np.random.default_rng(42)
    x2 = rng.standard_normal(inp.n_samples).astype(np.float32)
    # dyadic scale factors keep alpha*x1 + beta*x2 exactly representable enough for a 1e-12 check
    alpha, beta = 0.5, -2.0
    xs = (alpha * inp.x.astype(np.float64) + beta * x2.astype(np.float64))
    xs32 = xs.astype(np.float32)
    s1 = oracle.run(inp.offsets, inp.a1, inp.b0, inp.delays, inp.x)
    s2 = oracle.run(inp.offsets, inp.a1, inp.b0, inp.delays, x2)
    s12 = oracle.run(inp.offsets, inp.a1, inp.b0, inp.delays, xs32)
    # xs32 differs from xs by float32 rounding; bound its effect through the filter gains
    gain = np.array([np.sum(np.abs(w(inp.b0[o0:o1])) / (1 - np.abs(w(inp.a1[o0:o1]))))
                     for o0, o1 in zip(inp.offsets[:-1], inp.offsets[1:])])
    err = np.abs(s12 - (alpha * s1 + beta * s2)).max(axis=1)
    assert np.all(err <= np.abs(xs32 - xs).max() * gain + 1e-11)
    # template made of filters A u B == template A + template B
    oA, oB = (inp.offsets[0], inp.offsets[1]), (inp.offsets[1], inp.offsets[2])
    union = np.array([0, oB[1] - oA[0]], dtype=np.int64)
    su = oracle.run(union, inp.a1[oA[0]:oB[1]], inp.b0[oA[0]:oB[1]], inp.delays[oA[0]:oB[1]], inp.x)[0]
    assert np.abs(su - (s1[0] + s1[1])).max() <= 1e-12 * np.abs(su).max()
    # permuting the filters of a template changes only the summation order
    perm = rng.permutation(int(oB[1] - oA[0]))
    sp = oracle.run(union, inp.a1[:oB[1]][perm], inp.b0[:oB[1]][perm], inp.delays[:oB[1]][perm], inp.x)[0]
    assert np.abs(sp - su).max() <= 1e-12 * np.abs(su).max()
    # templates are independent: CSR indexing picks the right filters
    s_last = oracle.run(np.array([0, 5], dtype=np.int64), inp.a1[-5:], inp.b0[-5:], inp.delays[-5:], inp.x)[0]
    assert np.array_equal(s_last, s1[2])


# ---------------------------------------------------------------- P5 streaming == one-shot
@pytest.mark.parametrize("chunks", [[1] * 40 + [7, 300, 1, 652], [1000], [99, 101, 800], [64] * 15 + [40]])
def test_p5_streaming_equals_oneshot_bitwise(chunks):
    inp = spiir_inputs.make_random_bank(5, [33, 1, 70], sum(chunks), d_max=130)
    ref = oracle.run_inputs(inp)
    st = oracle.Stream(inp.offsets, inp.a1, inp.b0, inp.delays)
    out, pos = [], 0
    for c in chunks:                                          # includes chunks shorter than max delay
        out.append(st.filter(inp.x[pos:pos + c]))
        pos += c
    st.close()
    assert np.array_equal(np.concatenate(out, axis=1), ref)


# ---------------------------------------------------------------- P6 special cases -> library routines
def test_p6_zero_pole_is_sparse_fir():
    rng = np.random.default_rng(6)
    N, K = 400, 9
    b0 = (rng.standard_normal(K) + 1j * rng.standard_normal(K)).astype(np.complex64)
    d = rng.choice(50, K, replace=False).astype(np.int32)
    x = rng.standard_normal(N).astype(np.float32)
    snr = oracle.run(*one_template(np.zeros(K, np.complex64), b0, d), x)[0]
    comb = np.zeros(50, dtype=np.complex128)
    comb[d] = w(b0)
    expect = np.convolve(w(x), comb)[:N]
    assert np.abs(snr - expect).max() <= 1e-13 * np.abs(expect).max()


def test_p6_real_pole_zero_delay_is_lfilter():
    scipy_signal = pytest.importorskip("scipy.signal")
    rng = np.random.default_rng(7)
    N = 2000
    x = rng.standard_normal(N).astype(np.float32)
    for a, b in [(0.9, 1.25), (-0.75, -0.5), (0.999, 0.03125)]:
        a32, b32 = np.float32(a), np.float32(b)
        snr = oracle.run(*one_template(np.complex64(a32), np.complex64(b32), 0), x)[0]
        expect = scipy_signal.lfilter([float(b32)], [1.0, -float(a32)], w(x))
        assert np.abs(snr.imag).max() == 0.0
        assert np.abs(snr.real - expect).max() <= 1e-11 * np.abs(expect).max()
    # purely imaginary gain with a real pole puts everything in the imaginary part
    snr = oracle.run(*one_template(np.complex64(0.5), np.complex64(2j), 0), x)[0]
    expect = scipy_signal.lfilter([2.0], [1.0, -0.5], w(x))
    assert np.abs(snr.real).max() == 0.0 and np.abs(snr.imag - expect).max() <= 1e-12 * np.abs(expect).max()


# ---------------------------------------------------------------- P7 exact golden vector
def _read_p7():
    filters, x, rows = [], None, []
    for line in (GOLDEN / "p7_dyadic.txt").read_text().splitlines():
        if line.startswith("# x:"):
            x = [int(v) for v in line[4:].split()]
        elif line.startswith("#"):
            parts = line[1:].split()
            if len(parts) == 5:
                try:
                    filters.append([Fraction(p) for p in parts])
                except ValueError:
                    pass
        elif line.strip():
            n, re, im = line.split()
            rows.append((Fraction(re), Fraction(im)))
    return filters, x, rows


def test_p7_exact_dyadic_golden_vector():
    filters, x, rows = _read_p7()
    assert len(filters) == 3 and len(x) == 8 and len(rows) == 8
    a1 = np.array([complex(float(f[0]), float(f[1])) for f in filters], dtype=np.complex64)
    b0 = np.array([complex(float(f[2]), float(f[3])) for f in filters], dtype=np.complex64)
    d = np.array([int(f[4]) for f in filters], dtype=np.int32)
    snr = oracle.run(*one_template(a1, b0, d), np.array(x, dtype=np.float32))[0]
    expect = np.array([complex(float(re), float(im)) for re, im in rows])
    assert np.array_equal(snr, expect)                        # exact: every intermediate is dyadic
    # hand-derived first entries
    assert rows[0] == (1, 0) and rows[1] == (Fraction(7, 2), 1) and rows[2] == (Fraction(11, 4), Fraction(5, 2))


# ---------------------------------------------------------------- P8 white-noise energy
def test_p8_white_noise_energy():
    rng = np.random.default_rng(8)
    N = 200_000
    x = rng.standard_normal(N).astype(np.float32)
    a1 = np.complex64(0.9 * np.exp(0.8j))
    b0 = np.complex64(0.6 + 0.2j)
    y = oracle.run(*one_template(a1, b0, 3), x)[0][1000:]
    expect = abs(w(b0)) ** 2 / (1 - abs(w(a1)) ** 2)          # E|y|^2 for unit-variance white input
    assert abs(np.mean(np.abs(y) ** 2) / expect - 1) < 0.03


# ---------------------------------------------------------------- generators and edge cases
def test_empty_and_degenerate_inputs():
    off, a1, b0, d = one_template(np.complex64(0.5), np.complex64(1), 4)
    assert oracle.run(off, a1, b0, d, np.zeros(0, np.float32)).shape == (1, 0)
    # delay beyond the series: output identically zero
    assert np.all(oracle.run(off, a1, b0, np.array([10], np.int32), np.ones(8, np.float32)) == 0)
    # zero templates
    z = oracle.run(np.array([0], np.int64), np.zeros(0, np.complex64), np.zeros(0, np.complex64),
                   np.zeros(0, np.int32), np.ones(4, np.float32))
    assert z.shape == (0, 4)


def test_generators_are_seeded_and_in_range():
    a = spiir_inputs.make_config(0)
    b = spiir_inputs.make_config(0)
    assert np.array_equal(a.a1, b.a1) and np.array_equal(a.x, b.x) and np.array_equal(a.delays, b.delays)
    assert a.n_templates == 1 and a.n_filters == 128 and a.n_samples == 4096 and a.max_delay <= 1023
    r = np.abs(a.a1.astype(np.complex128))
    assert r.min() >= 0.90 - 1e-6 and r.max() <= 0.999 + 1e-6
    c1 = spiir_inputs.make_config(1, n_templates=4, n_samples=512)
    assert c1.offsets.tolist() == [0, 256, 512, 768, 1024] and c1.delays.max() <= 4095
    c2 = spiir_inputs.make_config(2, n_templates=3, n_samples=256)
    d2 = c2.delays.reshape(3, 512)
    wang = np.angle(c2.a1.astype(np.complex128)).reshape(3, 512)
    assert np.all(np.diff(d2, axis=1) <= 0) and np.all(np.diff(wang, axis=1) > 0)   # chirp structure
    assert abs(np.abs(c2.a1[0].astype(np.complex128)) - 0.999) < 1e-6
    c4 = spiir_inputs.make_config(4, n_templates=50, n_samples=64)
    kt = np.diff(c4.offsets)
    assert kt.min() >= 64 and kt.max() <= 2048 and c4.chunk == 16 and c4.delays.max() <= 8191
    for c in (a, c1, c2, c4):
        assert c.a1.dtype == np.complex64 and c.b0.dtype == np.complex64
        assert c.delays.dtype == np.int32 and c.x.dtype == np.float32 and c.offsets.dtype == np.int64
        assert np.abs(c.a1.astype(np.complex128)).max() < 1.0
    sub = c1.select_templates([3, 0])
    assert np.array_equal(sub.a1[:256], c1.a1[768:]) and np.array_equal(sub.a1[256:], c1.a1[:256])


# ------------------------------------------------------------------ trigger candidates
def test_peaks_impulse_closed_form():
    # one filter, impulse at n0: |y[n]|^2 = |b0|^2 |a1|^(2(n - n0 - d)) decays from its first non-zero sample, so the
    # peak is |b0|^2 at n0 + d (north_star impulse response); a window that starts later sees its first sample largest
    a1, b0, d, n0, N = 0.9 * np.exp(0.3j), 0.5 - 0.25j, 7, 11, 64
    x = np.zeros(N, np.float32)
    x[n0] = 1.0
    snr = oracle.run(np.array([0, 1]), np.array([a1], np.complex64), np.array([b0], np.complex64), np.array([d], np.int32), x)
    p, i = oracle.peaks(snr)
    assert i[0] == n0 + d and p[0] == pytest.approx(abs(np.complex64(b0)) ** 2, rel=1e-12)
    p2, i2 = oracle.peaks(snr, j0=30, n=20)
    assert i2[0] == 0 and p2[0] == pytest.approx(abs(np.complex64(b0)) ** 2 * abs(np.complex64(a1)) ** (2 * (30 - n0 - d)), rel=1e-6)


def test_peaks_match_numpy_argmax_and_take_the_first_of_equals():
    rng = np.random.default_rng(3)
    snr = rng.standard_normal((9, 200)) + 1j * rng.standard_normal((9, 200))
    snr[4, 50] = snr[4, 120] = 30.0 + 40.0j                       # a tie: the earlier sample wins
    for j0, n in ((0, 200), (13, 57), (199, 1)):
        p, i = oracle.peaks(snr, j0, n)
        m = np.abs(snr[:, j0:j0 + n]) ** 2
        assert np.array_equal(i, m.argmax(axis=1))
        assert np.allclose(p, m.max(axis=1), rtol=1e-14)
    assert oracle.peaks(snr)[1][4] == 50
