"""Pins of the float64 oracle against what the paper and the mathematics fix (no GPU).

Each test names the passage it pins.  A plausible mistake anywhere in oracle/spiir_oracle.c
(dropped term, wrong sign or index, transposed operand, off-by-one in the delay or in the
history carry) fails at least one of them.
"""
import numpy as np
import pytest
import scipy.signal

import oracle
from oracle import FilterOracle, MultirateOracle, ResampOracle, kaiser_taps


def c64(z):
    return np.asarray(z, dtype=np.complex64)


def one_filter(a1, b0, d, x):
    o = FilterOracle(c64([[a1]]), c64([[b0]]), np.array([[d]], np.int32))
    return o.filter(x)[0, 0]


A1 = np.complex64(0.97 * np.exp(0.31j))
B0 = np.complex64(0.4 - 1.3j)


# ---- O1, single filter: closed forms -----------------------------------------------------------

@pytest.mark.parametrize("d", [0, 1, 7, 63])
def test_impulse_response_closed_form_eq6(d):
    """PAPER.md:58-59 Eq. 6 with a delayed input (Eq. 7): impulse at 0 -> y_k = b0 a1^(k-d), k >= d."""
    n = 200
    x = np.zeros(n); x[0] = 1.0
    z = one_filter(A1, B0, d, x)
    k = np.arange(n)
    a, b = complex(A1), complex(B0)
    ref = np.where(k >= d, b * a ** np.maximum(k - d, 0), 0.0)
    assert np.allclose(z, ref, rtol=1e-12, atol=1e-15)
    assert np.all(z[:d] == 0)


def test_step_response_geometric_series():
    """Eq. 6 with x = 1: y_k = b0 (1 - a1^(k-d+1)) / (1 - a1) for k >= d."""
    n, d = 300, 5
    z = one_filter(A1, B0, d, np.ones(n))
    a, b = complex(A1), complex(B0)
    k = np.arange(n)
    ref = np.where(k >= d, b * (1 - a ** np.maximum(k - d + 1, 0)) / (1 - a), 0.0)
    assert np.allclose(z, ref, rtol=1e-10, atol=1e-14)


def test_sinusoid_steady_state():
    """Eq. 6 on x = cos(w k): steady state is the sum of the two complex-exponential responses
    b0 e^{-+i w d} e^{+-i w k} / (1 - a1 e^{-+i w})."""
    n, d, w = 4000, 11, 0.37
    a, b = complex(np.complex64(0.9 * np.exp(-0.8j))), complex(B0)
    k = np.arange(n)
    # x must be float32-representable?  no: the oracle takes doubles as they are.
    z = one_filter(np.complex64(a), B0, d, np.cos(w * k))
    resp = lambda s: b * np.exp(1j * s * w * (k - d)) / (1 - a * np.exp(-1j * s * w))
    ref = 0.5 * (resp(+1) + resp(-1))
    assert np.allclose(z[-500:], ref[-500:], rtol=1e-10, atol=1e-12)   # 0.9^3500 transient is gone


@pytest.mark.parametrize("d", [0, 3, 50])
def test_equals_scipy_lfilter(d):
    """Special case reducing to a library routine: y = lfilter([b0], [1, -a1], x delayed by d)."""
    rng = np.random.default_rng(7)
    x = rng.standard_normal(777)
    xd = np.concatenate([np.zeros(d), x])[: x.size]
    ref = scipy.signal.lfilter([complex(B0)], [1.0, -complex(A1)], xd.astype(complex))
    assert np.allclose(one_filter(A1, B0, d, x), ref, rtol=1e-12, atol=1e-14)


# ---- O1, banks: linearity, superposition, padding, brute force ---------------------------------

def small_bank(seed, T=3, L=6, dmax=40):
    rng = np.random.default_rng(seed)
    a1 = c64(rng.uniform(0.5, 0.999, (T, L)) * np.exp(1j * rng.uniform(0, 2 * np.pi, (T, L))))
    b0 = c64(rng.standard_normal((T, L)) + 1j * rng.standard_normal((T, L)))
    d = rng.integers(0, dmax + 1, (T, L)).astype(np.int32)
    return a1, b0, d


def test_linearity_in_x():
    a1, b0, d = small_bank(1)
    rng = np.random.default_rng(2)
    x1, x2 = rng.standard_normal(300), rng.standard_normal(300)
    z = lambda x: FilterOracle(a1, b0, d).filter(x)
    assert np.allclose(z(2.5 * x1 - 0.75 * x2), 2.5 * z(x1) - 0.75 * z(x2), rtol=1e-12, atol=1e-12)


def test_superposition_over_filters_eq8():
    """Eq. 8: the bank output is the sum of its L one-filter banks."""
    a1, b0, d = small_bank(3)
    x = np.random.default_rng(4).standard_normal(256)
    whole = FilterOracle(a1, b0, d).filter(x)
    parts = sum(FilterOracle(a1[:, l:l + 1], b0[:, l:l + 1], d[:, l:l + 1]).filter(x) for l in range(a1.shape[1]))
    assert np.allclose(whole, parts, rtol=1e-12, atol=1e-13)


def test_zero_coefficient_padding_changes_nothing():
    """inserting filters with zero coefficients leaves the result unchanged."""
    a1, b0, d = small_bank(5)
    x = np.random.default_rng(6).standard_normal(200)
    pad = lambda m, v: np.concatenate([m, np.full((m.shape[0], 3), v, m.dtype)], axis=1)
    z0 = FilterOracle(a1, b0, d).filter(x)
    z1 = FilterOracle(pad(a1, 0.9 + 0.1j), pad(b0, 0), pad(d, 17)).filter(x)
    assert np.array_equal(z0, z1)


def test_brute_force_convolution():
    """z = sum_l conv(x, h_l), h_l[n] = b0 a1^(n-d) [n >= d]  (Eq. 6/7/8 unrolled), tiny sizes."""
    T, L, n = 4, 8, 512
    a1, b0, d = small_bank(8, T, L, 100)
    x = np.random.default_rng(9).standard_normal(n)
    z = FilterOracle(a1, b0, d).filter(x)[0]
    for t in range(T):
        ref = np.zeros(n, complex)
        for l in range(L):
            h = np.zeros(n, complex)
            h[d[t, l]:] = complex(b0[t, l]) * complex(a1[t, l]) ** np.arange(n - d[t, l])
            ref += np.convolve(x, h)[:n]
        assert np.allclose(z[t], ref, rtol=1e-10, atol=1e-12)


def test_delay_and_template_indexing_not_transposed():
    """Each (template, filter) must use its own a1, b0 and d: distinct impulse responses per slot."""
    T, L = 3, 4
    a1, b0, d = small_bank(10, T, L, 20)
    x = np.zeros(64); x[0] = 1.0
    z = FilterOracle(a1, b0, d).filter(x)[0]
    k = np.arange(64)
    for t in range(T):
        ref = sum(np.where(k >= d[t, l], complex(b0[t, l]) * complex(a1[t, l]) ** np.maximum(k - d[t, l], 0), 0)
                  for l in range(L))
        assert np.allclose(z[t], ref, rtol=1e-12, atol=1e-14)


def test_streams_are_independent():
    a1, b0, d = small_bank(11)
    rng = np.random.default_rng(12)
    x = rng.standard_normal((2, 150))
    both = FilterOracle(a1, b0, d, n_streams=2).filter(x)
    for s in range(2):
        assert np.array_equal(both[s], FilterOracle(a1, b0, d).filter(x[s])[0])


# ---- O1 streaming: block partition == one long run (bitwise) ------------------------------------

@pytest.mark.parametrize("cuts", [[1] * 40, [7, 1, 100, 33, 259], [400], [3, 397], [200, 200]])
def test_block_streaming_equals_one_run(cuts):
    a1, b0, d = small_bank(13, dmax=60)       # blocks shorter and longer than d_max = 60
    n = sum(cuts)
    x = np.random.default_rng(14).standard_normal(n)
    ref = FilterOracle(a1, b0, d).filter(x)
    o = FilterOracle(a1, b0, d)
    pos, outs = 0, []
    for c in cuts:
        outs.append(o.filter(x[pos:pos + c])); pos += c
    assert np.array_equal(np.concatenate(outs, axis=2), ref)
    o.reset()
    assert np.array_equal(o.filter(x), ref)


@pytest.mark.parametrize("cuts", [[23, 5, 41, 130, 1], [17] * 9, [3, 90, 2, 58]])
def test_two_streams_streamed_equal_each_stream_alone(cuts):
    """Per-stream history carry (hist + s*D) and per-stream state: S = 2 streamed over ragged blocks,
    some shorter than d_max = 60, must equal (bitwise) the S = 1 oracle run on each stream alone in
    ONE call, and the S = 2 one-call run.  Mixing up the two histories or states fails this."""
    a1, b0, d = small_bank(15, dmax=60)
    n = sum(cuts)
    x = np.random.default_rng(16).standard_normal((2, n))
    o = FilterOracle(a1, b0, d, n_streams=2)
    pos, outs = 0, []
    for c in cuts:
        outs.append(o.filter(x[:, pos:pos + c])); pos += c
    got = np.concatenate(outs, axis=2)
    assert np.array_equal(got, FilterOracle(a1, b0, d, n_streams=2).filter(x))
    for s in range(2):
        assert np.array_equal(got[s], FilterOracle(a1, b0, d).filter(x[s])[0])
    assert not np.array_equal(got[0], got[1])


# ---- O4 taps ---------------------------------------------------------------------------------

def test_taps_match_numpy_kaiser_times_sinc():
    """DESIGN.md O4 / PAPER.md:84 'Kaiser-window-tapered low-pass filter'."""
    N, beta, fc = 192, 5.0, 0.25
    h64, h32 = kaiser_taps(N, beta, fc)
    n = np.arange(N)
    ref = np.kaiser(N, beta) * 2 * fc * np.sinc(2 * fc * (n - (N - 1) / 2))
    ref /= ref.sum()
    assert np.allclose(h64, ref, rtol=1e-12, atol=1e-16)
    assert np.array_equal(h32, ref.astype(np.float32)) or np.max(np.abs(h32 - ref)) < 1e-9
    assert np.allclose(h64, h64[::-1], rtol=0, atol=1e-16)                  # symmetric
    assert abs(h64.sum() - 1) < 1e-14
    assert abs(h64[0::2].sum() - 0.5) < 1e-3 and abs(h64[1::2].sum() - 0.5) < 1e-3
    assert np.allclose(h64[1::2], h64[0::2][::-1], atol=1e-16)              # odd branch = reversed even branch


def test_taps_frequency_response():
    """Reading R3: pass band flat to 0.20 cycles/sample, -6 dB at 0.25, >= 50 dB down beyond 0.30."""
    h64, _ = kaiser_taps()
    f = np.linspace(0, 0.5, 2001)
    Hf = np.abs(np.exp(-2j * np.pi * np.outer(f, np.arange(192))) @ h64)
    assert np.max(np.abs(Hf[f <= 0.20] - 1)) < 1e-3
    assert abs(Hf[np.argmin(np.abs(f - 0.25))] - 0.5) < 5e-3
    assert np.max(Hf[f >= 0.30]) < 10 ** (-50 / 20)


# ---- O2 / O3 resamplers --------------------------------------------------------------------------

def test_down2_equals_numpy_convolve_stride():
    _, h32 = kaiser_taps()
    u = np.random.default_rng(20).standard_normal((3, 1000))
    out = ResampOracle("down", 3).down(u)
    for r in range(3):
        ref = np.convolve(u[r], h32.astype(np.float64))[0:1000:2]            # v[m] = (h * u)[2m]
        assert np.allclose(out[r], ref, rtol=1e-12, atol=1e-14)


def test_up2_equals_zero_stuff_convolve():
    _, h32 = kaiser_taps()
    rng = np.random.default_rng(21)
    v = rng.standard_normal((2, 300)) + 1j * rng.standard_normal((2, 300))
    out = ResampOracle("up", 2).up(v)
    for r in range(2):
        stuffed = np.zeros(600, complex); stuffed[0::2] = v[r]
        ref = 2 * np.convolve(stuffed, h32.astype(np.float64))[:600]
        assert np.allclose(out[r], ref, rtol=1e-12, atol=1e-14)


@pytest.mark.parametrize("n_taps,beta", [(32, 5.0), (384, 10.0), (64, 7.0)])
def test_resamplers_other_tap_counts_equal_numpy_convolve(n_taps, beta):
    """384 taps down / 32 taps up are the paper's own filter lengths; the resamplers
    must stay the plain convolution for any even N (history N-1 / N/2-1, streamed in ragged blocks)."""
    _, h32 = kaiser_taps(n_taps, beta, 0.25)
    h = h32.astype(np.float64)
    rng = np.random.default_rng(n_taps)
    u = rng.standard_normal((2, 900))
    v = rng.standard_normal((2, 450)) + 1j * rng.standard_normal((2, 450))
    od = ResampOracle("down", 2, n_taps=n_taps, beta=beta)
    ou = ResampOracle("up", 2, n_taps=n_taps, beta=beta)
    got_d = np.concatenate([od.down(u[:, a:b]) for a, b in ((0, 2), (2, 300), (300, 900))], axis=1)
    got_u = np.concatenate([ou.up(v[:, a:b]) for a, b in ((0, 1), (1, 7), (7, 450))], axis=1)
    for r in range(2):
        assert np.allclose(got_d[r], np.convolve(u[r], h)[0:900:2], rtol=1e-12, atol=1e-14)
        stuffed = np.zeros(900, complex); stuffed[0::2] = v[r]
        assert np.allclose(got_u[r], 2 * np.convolve(stuffed, h)[:900], rtol=1e-12, atol=1e-14)


def test_up2_accumulate_adds():
    rng = np.random.default_rng(22)
    v = rng.standard_normal((2, 64)) + 1j * rng.standard_normal((2, 64))
    base = rng.standard_normal((2, 128)) + 1j * rng.standard_normal((2, 128))
    plain = ResampOracle("up", 2).up(v)
    acc = ResampOracle("up", 2).up(v, out=base.copy())
    assert np.allclose(acc, base + plain, rtol=1e-14, atol=1e-15)


@pytest.mark.parametrize("cuts", [[2] * 30, [64, 2, 190, 500, 44], [800]])
def test_resamplers_stream(cuts):
    n = sum(cuts)
    rng = np.random.default_rng(23)
    u = rng.standard_normal((2, n))
    v = rng.standard_normal((2, n)) + 1j * rng.standard_normal((2, n))
    ref_d, ref_u = ResampOracle("down", 2).down(u), ResampOracle("up", 2).up(v)
    od, ou = ResampOracle("down", 2), ResampOracle("up", 2)
    pos, outs_d, outs_u = 0, [], []
    for c in cuts:
        outs_d.append(od.down(u[:, pos:pos + c])); outs_u.append(ou.up(v[:, pos:pos + c])); pos += c
    assert np.array_equal(np.concatenate(outs_d, axis=1), ref_d)
    assert np.array_equal(np.concatenate(outs_u, axis=1), ref_u)


def test_dc_preserved_and_tone_round_trip():
    """north_star (e): DC and low-frequency sinusoids survive decimate-then-interpolate, delayed by
    N-1 = 191 high-rate samples (reading R4), within the pass-band ripple; a tone above the new
    Nyquist is attenuated >= 50 dB by the decimator."""
    n = 4096
    k = np.arange(n)
    down, up = ResampOracle("down", 1), ResampOracle("up", 1)
    dc = up.up(down.down(np.ones(n)).astype(complex))[0]
    assert np.max(np.abs(dc[400:] - 1)) < 2e-6          # float32-rounded taps: branch sums = 1 +- 1e-7
    for f in (0.01, 0.05, 0.11, 0.20):
        down.reset(); up.reset()
        x = np.cos(2 * np.pi * f * k)
        y = up.up(down.down(x).astype(complex))[0].real
        assert np.max(np.abs(y[600:] - x[600 - 191:n - 191])) < 2e-3, f
    down.reset()
    hi = down.down(np.cos(2 * np.pi * 0.31 * k))[0]
    assert np.max(np.abs(hi[200:])) < 10 ** (-50 / 20)


# ---- O5 multirate ---------------------------------------------------------------------------------

def mr_banks(seed, T, Ls, dmaxs):
    return [small_bank(seed + i, T, L, dm) for i, (L, dm) in enumerate(zip(Ls, dmaxs))]


def test_multirate_single_rate_is_plain_filter():
    banks = mr_banks(30, 2, [5], [30])
    x = np.random.default_rng(31).standard_normal(256)
    assert np.array_equal(MultirateOracle(banks).filter(x), FilterOracle(*banks[0]).filter(x))


def test_multirate_cascade_equals_direct_to_base_rate():
    """Reading R6: by linearity the cascade equals upsampling every rate's SNR straight to the base
    rate through its own chain of up-by-2 stages and summing."""
    T, n = 2, 512
    banks = mr_banks(32, T, [3, 4, 5], [20, 20, 10])
    x = np.random.default_rng(33).standard_normal(n)
    got = MultirateOracle(banks).filter(x)
    xs = [x[None, :]]
    for h in (1, 2):
        xs.append(ResampOracle("down", 1).down(xs[-1]))
    total = np.zeros((T, n), complex)
    for h in range(3):
        z = FilterOracle(*banks[h]).filter(xs[h])[0]
        for _ in range(h):
            z = ResampOracle("up", T).up(z)
        total += z
    assert np.allclose(got[0], total, rtol=1e-9, atol=1e-12)


def test_multirate_streams_in_blocks():
    banks = mr_banks(34, 2, [3, 2, 4], [15, 9, 6])
    x = np.random.default_rng(35).standard_normal(1024)
    ref = MultirateOracle(banks).filter(x)
    o = MultirateOracle(banks)
    got = np.concatenate([o.filter(x[i:i + 256]) for i in range(0, 1024, 256)], axis=2)
    assert np.array_equal(got, ref)


def test_multirate_two_streams_streamed_equal_each_stream_alone():
    """MultirateOracle(n_streams=2): the rows = S*T reshape of the up cascade and the per-stream FIR /
    bank histories, streamed over ragged blocks (multiples of 2^(H-1) = 4, some shorter than the
    delays and FIR histories), equal the S = 1 oracle on each stream alone in one call (bitwise)."""
    banks = mr_banks(36, 3, [3, 2, 4], [40, 25, 12])
    n = 1024
    x = np.random.default_rng(37).standard_normal((2, n))
    o = MultirateOracle(banks, n_streams=2)
    cuts, pos, outs = [4, 60, 256, 8, 696], 0, []
    for c in cuts:
        outs.append(o.filter(x[:, pos:pos + c])); pos += c
    got = np.concatenate(outs, axis=2)
    assert got.shape == (2, 3, n)
    for s in range(2):
        assert np.array_equal(got[s], MultirateOracle(banks).filter(x[s])[0])
    assert not np.array_equal(got[0], got[1])


def test_multirate_separate_down_up_taps_cascade_equals_direct():
    """different filters per direction (384-tap down, 32-tap up).  Same linearity pin
    as above with the two tap sets passed separately."""
    T, n = 2, 512
    banks = mr_banks(38, T, [3, 4], [20, 10])
    x = np.random.default_rng(39).standard_normal(n)
    kw = dict(n_taps_down=384, beta_down=10.0, n_taps_up=32, beta_up=5.0)
    got = MultirateOracle(banks, **kw).filter(x)
    x1 = ResampOracle("down", 1, n_taps=384, beta=10.0).down(x[None, :])
    z0 = FilterOracle(*banks[0]).filter(x)[0]
    z1 = ResampOracle("up", T, n_taps=32, beta=5.0).up(FilterOracle(*banks[1]).filter(x1)[0])
    assert np.allclose(got[0], z0 + z1, rtol=1e-12, atol=1e-14)


def test_oracle_reports_threads():
    assert oracle.num_threads() >= 1
