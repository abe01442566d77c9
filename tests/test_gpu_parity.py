"""GPU parity: the CUDA path (through the C ABI) against the float64 oracle, element by element,
on the same seeded inputs.  Tolerances are BASELINE.json north_star's (tests/_util.py).

Sizes: cut-down configs the oracle finishes in seconds (several tiles, ragged tails), plus the
full BASELINE.json sizes in the launch configuration bench.py times, checked on sampled templates
the oracle computes one by one (every template is an independent unit).
"""
import numpy as np
import pytest

from _util import ParityAccumulator, assert_parity, stream_gpu_plan, stream_oracle

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sp():
    import paper_1702_02256_b200 as sp
    sp.lib()                       # fails loudly when the extension is missing
    return sp


@pytest.fixture(scope="module")
def oracle_mod():
    import oracle
    return oracle


def _inputs():
    from paper_1702_02256_b200 import inputs
    return inputs


def _bank_tuple(b):
    return (b.a1, b.b0, b.delays)


# ------------------------------------------------------------------------------------------------
# config 0: 16 x 128, one block of 4096, zero initial state -- plain and time-chunked geometry
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("time_chunks", [1, 0, 7])
def test_config0_full(sp, oracle_mod, time_chunks):
    w = _inputs().config(0)
    b = w.banks[0]
    plan = sp.Plan(b.a1, b.b0, b.delays, b.rate_hz, max_block=w.block, time_chunks=time_chunks)
    info = plan.launch_info(w.block)
    if time_chunks == 1:
        assert info["time_chunks"] == 1 and info["launches"] == 1
    if time_chunks == 0:
        assert info["time_chunks"] > 1 and info["launches"] == 3      # under-occupied bank -> chunked scan
    x = [w.strain(0)]
    z = stream_gpu_plan(plan, x)
    ref = stream_oracle(oracle_mod.FilterOracle(b.a1, b.b0, b.delays), x)
    assert z.shape == (1, 16, 4096)
    assert_parity(z, ref, f"cfg0 chunks={time_chunks}")


# ------------------------------------------------------------------------------------------------
# config 1: many-filter regime, streamed blocks with carried state and history
# ------------------------------------------------------------------------------------------------
def test_config1_cut_streamed(sp, oracle_mod):
    w = _inputs().config(1, n_templates=40, n_blocks=4)
    b = w.banks[0]
    plan = sp.Plan(b.a1, b.b0, b.delays, b.rate_hz, max_block=w.block, time_chunks=1)
    xs = [w.strain(i) for i in range(4)]
    z = stream_gpu_plan(plan, xs)
    ref = stream_oracle(oracle_mod.FilterOracle(b.a1, b.b0, b.delays), xs)
    assert_parity(z, ref, "cfg1 cut")


def test_config1_full_size_sampled(sp, oracle_mod):
    """Full 1024 x 256 bank in the geometry bench.py times; oracle on sampled templates."""
    w = _inputs().config(1)
    b = w.banks[0]
    plan = sp.Plan(b.a1, b.b0, b.delays, b.rate_hz, max_block=w.block)
    info = plan.launch_info(w.block)
    assert info["F"] == 8 and info["lanes_per_template"] == 32 and info["time_chunks"] == 1
    xs = [w.strain(i) for i in range(3)]
    z = stream_gpu_plan(plan, xs)
    idx = np.array([0, 1, 6, 7, 8, 511, 512, 777, 1017, 1022, 1023])
    ref = stream_oracle(oracle_mod.FilterOracle(b.a1[idx], b.b0[idx], b.delays[idx]), xs)
    assert_parity(z[:, idx], ref, "cfg1 full sampled")


def test_half_warp_per_template_mapping(sp, oracle_mod):
    """Banks with >= 2368 templates: 32..64 filters put four templates in a warp (8 lanes each), 65..128 two (16 lanes)."""
    for L in (32, 40, 64, 72, 128):
        w = _inputs().config(1, n_templates=2400, n_filters=L)
        b = w.banks[0]
        plan = sp.Plan(b.a1, b.b0, b.delays % 300, b.rate_hz, max_block=256)
        info = plan.launch_info(256)
        lpt = 8 if L <= 64 else 16
        assert info["lanes_per_template"] == lpt and info["F"] == (L + lpt - 1) // lpt
        rng = np.random.default_rng(L)
        xs = [rng.standard_normal((1, n)).astype(np.float32) for n in (256, 37, 160)]
        z = stream_gpu_plan(plan, xs)
        idx = np.array([0, 1, 2, 3, 1199, 1200, 2397, 2398, 2399])
        ref = stream_oracle(oracle_mod.FilterOracle(b.a1[idx], b.b0[idx], (b.delays % 300)[idx]), xs)
        assert_parity(z[:, idx], ref, f"LPT16 L={L}")


# ------------------------------------------------------------------------------------------------
# config 2: few-filter sweep, 4096 templates, 256-sample blocks
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L", [1, 2, 4, 8, 16, 32])
def test_config2_few_filter(sp, oracle_mod, L):
    w = _inputs().config(2, n_filters=L, n_blocks=6)
    b = w.banks[0]
    plan = sp.Plan(b.a1, b.b0, b.delays, b.rate_hz, max_block=w.block)
    xs = [w.strain(i) for i in range(6)]
    z = stream_gpu_plan(plan, xs)
    ref = stream_oracle(oracle_mod.FilterOracle(b.a1, b.b0, b.delays), xs)
    assert z.shape == (1, 4096, 6 * 256)
    assert_parity(z, ref, f"cfg2 L={L}")


@pytest.mark.parametrize("T,L,S,chunks,blocks", [
    (70, 1, 1, 0, (256, 256, 37, 1, 64, 300)),          # partially filled last group, ragged blocks, plain fallback below 64
    (33, 4, 2, 0, (512, 100, 512)),                      # two streams
    (20, 7, 1, 5, (1000, 333)),                          # two lanes per template, forced chunk count
    (9, 13, 1, 16, (2048, 2048)),                        # four lanes per template
    (5, 29, 1, 3, (700, 90, 700)),                       # eight lanes per template
    (40, 2, 1, 0, (20000, 4000)),                        # block longer than the shared-memory window: several time tiles
])
def test_in_cta_time_scan(sp, oracle_mod, T, L, S, chunks, blocks):
    """Row a7 for the few-filter mappings: the time chunks are the warps of one CTA (spiir_filter_scan_kernel)."""
    w = _inputs().config(2, n_templates=T, n_filters=L)
    b = w.banks[0]
    delays = b.delays.copy()
    delays.flat[0] = 0
    delays.flat[-1] = 255
    plan = sp.Plan(b.a1, b.b0, delays, b.rate_hz, n_streams=S, max_block=max(blocks), time_chunks=chunks)
    info = plan.launch_info(max(blocks))
    assert info["launches"] == 1 and info["time_chunks"] > 1, info
    rng = np.random.default_rng(T * 100 + L)
    xs = [rng.standard_normal((S, n)).astype(np.float32) for n in blocks]
    z = stream_gpu_plan(plan, xs)
    ref = stream_oracle(oracle_mod.FilterOracle(b.a1, b.b0, delays, S), xs)
    assert_parity(z, ref, f"in-CTA scan T={T} L={L} S={S}")
    plain = stream_gpu_plan(sp.Plan(b.a1, b.b0, delays, b.rate_hz, n_streams=S, max_block=max(blocks), time_chunks=1), xs)
    assert_parity(plain, ref, "plain")


def test_phase_word_has_one_reader_per_cta(sp, oracle_mod):
    """Regression (found by a randomised parity run): every thread used to read the ping-pong phase word itself, so a slow
    warp of a late CTA could read it after the launch's last share had landed and take the NEXT phase -- the wrong history
    buffer for its templates, about one fresh plan in four with this shape (450 CTAs of 5 warps, three streams).  Twelve
    fresh plans, one block each, every output compared."""
    import torch
    rng = np.random.default_rng(5)
    T, L, S, n = 600, 24, 3, 1130
    mag, arg = rng.uniform(0.5, 0.9999, (T, L)), rng.uniform(0, 2 * np.pi, (T, L))
    a1 = (mag * np.exp(1j * arg)).astype(np.complex64)
    b0 = (1e-3 * (rng.standard_normal((T, L)) + 1j * rng.standard_normal((T, L)))).astype(np.complex64)
    d = rng.integers(0, 101, (T, L)).astype(np.int32)
    x = rng.standard_normal((S, n)).astype(np.float32)
    ref = oracle_mod.FilterOracle(a1, b0, d, S).filter(x)
    xd = torch.from_numpy(x).cuda()
    for trial in range(12):
        plan = sp.Plan(a1, b0, d, 4096, n_streams=S, max_block=2048)
        z = plan.filter(xd).cpu().numpy()
        hist = plan.get_state()[1].cpu().numpy()
        plan.close()
        assert_parity(z, ref, f"fresh plan {trial}")
        np.testing.assert_array_equal(hist, x[:, -hist.shape[1]:])


def test_config2_bulk_call_sampled(sp, oracle_mod):
    """configs[2] as ONE call of 64 x 256 = 16384 samples (the bulk shape bench.py times), L = 1 and 4: full bank on the
    GPU, the oracle on templates spread over every CTA (first and last included)."""
    import torch
    for L in (1, 4):
        w = _inputs().config(2, n_filters=L)
        b = w.banks[0]
        n = 64 * w.block
        plan = sp.Plan(b.a1, b.b0, b.delays, b.rate_hz, max_block=n)
        xs = [np.concatenate([w.strain(k * 64 + i) for i in range(64)], -1) for k in range(2)]
        idx = np.unique(np.concatenate([np.arange(0, 4096, 37), [31, 32, 4095]]))
        orc = oracle_mod.FilterOracle(b.a1[idx], b.b0[idx], b.delays[idx])
        acc = ParityAccumulator()
        for x in xs:
            z = plan.filter(torch.from_numpy(x).cuda())
            acc.add(z[:, torch.from_numpy(idx).cuda()].cpu().numpy(), orc.filter(x))
        acc.check(f"cfg2 bulk L={L}")


# ------------------------------------------------------------------------------------------------
# config 3: multirate, 7 rates, 192-tap Kaiser resamplers, cascade accumulation
# ------------------------------------------------------------------------------------------------
def test_config3_multirate_cut(sp, oracle_mod):
    w = _inputs().config(3, n_templates=24, n_blocks=3)
    banks = [_bank_tuple(b) for b in w.banks]
    mr = sp.MultiratePlan(banks, [b.rate_hz for b in w.banks], max_block=w.block)
    xs = [w.strain(i) for i in range(3)]
    z = stream_gpu_plan(mr, xs)
    ref = stream_oracle(oracle_mod.MultirateOracle(banks), xs)
    assert_parity(z, ref, "cfg3 cut")


def test_config3_full_size_sampled(sp, oracle_mod):
    w = _inputs().config(3)
    banks = [_bank_tuple(b) for b in w.banks]
    mr = sp.MultiratePlan(banks, [b.rate_hz for b in w.banks], max_block=w.block)
    xs = [w.strain(i) for i in range(2)]
    z = stream_gpu_plan(mr, xs)
    idx = np.array([0, 3, 500, 1023])
    ref = stream_oracle(oracle_mod.MultirateOracle([(a[idx], b_[idx], d[idx]) for (a, b_, d) in banks]), xs)
    assert_parity(z[:, idx], ref, "cfg3 full sampled")


def test_multirate_small_blocks(sp, oracle_mod):
    """Blocks of 64 and 192 base-rate samples (one / three samples at 64 Hz)."""
    w = _inputs().config(3, n_templates=8)
    banks = [_bank_tuple(b) for b in w.banks]
    mr = sp.MultiratePlan(banks, [b.rate_hz for b in w.banks], max_block=4096)
    rng = np.random.default_rng(7)
    xs = [rng.standard_normal((1, n)).astype(np.float32) for n in (64, 192, 4096, 128, 1024)]
    z = stream_gpu_plan(mr, xs)
    ref = stream_oracle(oracle_mod.MultirateOracle(banks), xs)
    assert_parity(z, ref, "multirate ragged blocks")


# ------------------------------------------------------------------------------------------------
# config 4: two detectors x 16384 templates x 256 filters at 2048 Hz
# ------------------------------------------------------------------------------------------------
def test_config4_cut_two_streams(sp, oracle_mod):
    w = _inputs().config(4, n_templates=20, n_blocks=3)
    b = w.banks[0]
    plan = sp.Plan(b.a1, b.b0, b.delays, b.rate_hz, n_streams=2, max_block=w.block, time_chunks=1)
    xs = [w.strain(i) for i in range(3)]
    z = stream_gpu_plan(plan, xs)
    ref = stream_oracle(oracle_mod.FilterOracle(b.a1, b.b0, b.delays, 2), xs)
    assert z.shape == (2, 20, 3 * 2048)
    assert_parity(z, ref, "cfg4 cut")


def test_config4_full_size_sampled(sp, oracle_mod):
    import torch
    w = _inputs().config(4)
    b = w.banks[0]
    plan = sp.Plan(b.a1, b.b0, b.delays, b.rate_hz, n_streams=2, max_block=w.block)
    idx = np.array([0, 1, 8191, 8192, 12345, 16383])
    ref_o = oracle_mod.FilterOracle(b.a1[idx], b.b0[idx], b.delays[idx], 2)
    out = torch.empty((2, w.n_templates, w.block), dtype=torch.complex64, device="cuda")
    zs, rs = [], []
    for i in range(2):
        x = w.strain(i)
        plan.filter(torch.from_numpy(x).cuda(), out)
        zs.append(out[:, torch.from_numpy(idx).cuda()].cpu().numpy())
        rs.append(ref_o.filter(x))
    assert_parity(np.concatenate(zs, -1), np.concatenate(rs, -1), "cfg4 full sampled")


# ------------------------------------------------------------------------------------------------
# properties that hold at any size
# ------------------------------------------------------------------------------------------------
def test_block_partition_equals_one_run(sp):
    """Streaming check (d) of north_star on the GPU side: ragged partition == one long call,
    to float32 rounding (the chunked path sums in a different order)."""
    w = _inputs().config(1, n_templates=12)
    b = w.banks[0]
    rng = np.random.default_rng(11)
    x = rng.standard_normal((1, 6000)).astype(np.float32)
    one = stream_gpu_plan(sp.Plan(b.a1, b.b0, b.delays, max_block=6000, time_chunks=1), [x])
    cuts = [0, 1, 18, 1019, 1020, 3333, 6000]
    parts = [x[:, cuts[i]:cuts[i + 1]] for i in range(len(cuts) - 1)]
    many = stream_gpu_plan(sp.Plan(b.a1, b.b0, b.delays, max_block=6000, time_chunks=1), parts)
    np.testing.assert_array_equal(one, many)       # same kernel, same order of operations: bit-exact
    chunked = stream_gpu_plan(sp.Plan(b.a1, b.b0, b.delays, max_block=6000, time_chunks=5), [x])
    assert_parity(chunked, one.astype(np.complex128), "chunked vs plain")


def test_deterministic(sp):
    w = _inputs().config(0)
    b = w.banks[0]
    x = [w.strain(0)]
    z1 = stream_gpu_plan(sp.Plan(b.a1, b.b0, b.delays, max_block=4096), x)
    z2 = stream_gpu_plan(sp.Plan(b.a1, b.b0, b.delays, max_block=4096), x)
    np.testing.assert_array_equal(z1, z2)


def test_zero_padding_changes_nothing(sp, oracle_mod):
    """padding a bank with zero-coefficient filters leaves the SNR unchanged."""
    w = _inputs().config(0, n_templates=6, n_filters=37)
    b = w.banks[0]
    pad = 64 - 37
    a1 = np.concatenate([b.a1, np.zeros((6, pad), np.complex64)], 1)
    b0 = np.concatenate([b.b0, np.zeros((6, pad), np.complex64)], 1)
    d = np.concatenate([b.delays, np.zeros((6, pad), np.int32)], 1)
    x = [w.strain(0)[:, :1500]]
    z37 = stream_gpu_plan(sp.Plan(b.a1, b.b0, b.delays, max_block=1500, time_chunks=1), x)
    z64 = stream_gpu_plan(sp.Plan(a1, b0, d, max_block=1500, time_chunks=1), x)
    ref = stream_oracle(oracle_mod.FilterOracle(b.a1, b.b0, b.delays), x)
    assert_parity(z37, ref, "L=37")
    assert_parity(z64, ref, "L=37 padded to 64")


@pytest.mark.parametrize("T,L", [(5, 5), (3, 513 // 3), (33, 3), (7, 20), (2, 300), (1, 512), (9, 96)])
def test_odd_shapes(sp, oracle_mod, T, L):
    """Filter counts from PAPER.md:104 (5 filters; several small templates per warp) and banks that
    do not fill their last warp."""
    w = _inputs().config(0, n_templates=T, n_filters=L)
    b = w.banks[0]
    rng = np.random.default_rng(T * 1000 + L)
    xs = [rng.standard_normal((1, n)).astype(np.float32) for n in (700, 33, 1)]
    z = stream_gpu_plan(sp.Plan(b.a1, b.b0, b.delays, max_block=700, time_chunks=1), xs)
    ref = stream_oracle(oracle_mod.FilterOracle(b.a1, b.b0, b.delays), xs)
    assert_parity(z, ref, f"T={T} L={L}")


@pytest.mark.parametrize("T,L", [(3, 513), (5, 544), (2, 1024), (9, 700), (1, 2048)])
def test_templates_of_more_than_512_filters(sp, oracle_mod, T, L):
    """PAPER.md:104 (513 filters -> 544 threads of one block), PAPER.md:233 (1024 filters per template at one rate):
    a template spans several warps of one CTA, partial sums meet in shared memory."""
    w = _inputs().config(0, n_templates=T, n_filters=L)
    b = w.banks[0]
    m = sp.spiir_host_lane_mapping(L)
    assert m["warps_per_template"] >= 2 and m["F"] * 32 * m["warps_per_template"] >= L
    rng = np.random.default_rng(T * 10000 + L)
    xs = [rng.standard_normal((1, n)).astype(np.float32) for n in (900, 33, 1, 600)]
    z = stream_gpu_plan(sp.Plan(b.a1, b.b0, b.delays, max_block=900, time_chunks=1), xs)
    ref = stream_oracle(oracle_mod.FilterOracle(b.a1, b.b0, b.delays), xs)
    assert_parity(z, ref, f"T={T} L={L}")
    if L == 513:                                                  # also through the chunked scan
        zc = stream_gpu_plan(sp.Plan(b.a1, b.b0, b.delays, max_block=900, time_chunks=3), xs)
        assert_parity(zc, ref, f"T={T} L={L} chunked")


def test_filter_count_limit(sp):
    w = _inputs().config(0, n_templates=1, n_filters=2049)
    b = w.banks[0]
    with pytest.raises(sp.SpiirError) as e:
        sp.Plan(b.a1, b.b0, b.delays)
    assert e.value.status == sp.SPIIR_EUNSUPPORTED


def _ragged_bank(counts, seed, d_max=300):
    """Flat CSR arrays of a bank whose template t has counts[t] filters (configs[0] distributions), plus the same
    bank padded with b0 = 0 filters to the longest template: the oracle's way to express a ragged bank (F6)."""
    inp = _inputs()
    Lmax = max(counts)
    full = inp.make_bank((77, seed), len(counts), Lmax, 4096, 0.9, 0.9999, d_max)
    off = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
    a1 = np.concatenate([full.a1[t, :c] for t, c in enumerate(counts)])
    b0 = np.concatenate([full.b0[t, :c] for t, c in enumerate(counts)])
    d = np.concatenate([full.delays[t, :c] for t, c in enumerate(counts)])
    pa1, pb0, pd = full.a1.copy(), full.b0.copy(), full.delays.copy()
    for t, c in enumerate(counts):
        pa1[t, c:] = 0; pb0[t, c:] = 0; pd[t, c:] = 0
    return (a1, b0, d, off), (pa1, pb0, pd)


@pytest.mark.parametrize("counts", [[5, 513, 1024], [5, 5, 5, 5, 17, 1, 300, 32, 31, 33, 256, 2, 700, 64, 5, 128],
                                    [7] * 40 + [200] * 3 + [1] * 9])
def test_ragged_bank(sp, oracle_mod, counts):
    """spiir_plan_create_ragged (templates of 5, 513 filters; several small templates per warp):
    per-template filter counts, output rows in the caller's template order, state in CSR order."""
    import torch
    (a1, b0, d, off), (pa1, pb0, pd) = _ragged_bank(counts, len(counts))
    plan = sp.Plan.ragged(a1, b0, d, off, max_block=700, time_chunks=1)
    assert plan.T == len(counts) and plan.n_filters_total == sum(counts)
    rng = np.random.default_rng(sum(counts))
    xs = [rng.standard_normal((1, n)).astype(np.float32) for n in (700, 19, 400)]
    z = stream_gpu_plan(plan, xs)
    ref = stream_oracle(oracle_mod.FilterOracle(pa1, pb0, pd), xs)
    assert z.shape == (1, len(counts), 1119)
    assert_parity(z, ref, f"ragged {counts[:4]}...")
    # resume state in CSR order: filter i of template t is y of the one-filter oracle (t, i) after the run
    y, hist = plan.get_state()
    y = y.cpu().numpy()[0]
    xall = np.concatenate(xs, -1)
    np.testing.assert_array_equal(hist.cpu().numpy()[0], xall[0, -plan.history_len:])
    for t in (0, len(counts) - 1, len(counts) // 2):
        for i in {0, counts[t] - 1}:
            k = off[t] + i
            one = oracle_mod.FilterOracle(a1[k:k + 1][None], b0[k:k + 1][None], d[k:k + 1][None]).filter(xall)[0, 0, -1]
            assert abs(y[k] - one) <= 2e-5 * max(abs(one), 1e-6), (t, i)
    # a second ragged plan given that state continues the stream bit-exactly
    x2 = rng.standard_normal((1, 300)).astype(np.float32)
    z2 = plan.filter(torch.from_numpy(x2).cuda()).cpu().numpy()
    fresh = sp.Plan.ragged(a1, b0, d, off, max_block=700, time_chunks=1)
    yy, hh = torch.from_numpy(y[None]).cuda(), hist
    fresh.set_state(yy, hh)
    np.testing.assert_array_equal(fresh.filter(torch.from_numpy(x2).cuda()).cpu().numpy(), z2)


def test_degenerate_delays_and_alignment(sp, oracle_mod):
    """d = 0 everywhere; delays beyond the block length; x pointer not 16-byte aligned (no TMA)."""
    import torch
    w = _inputs().config(0, n_templates=4, n_filters=64)
    b = w.banks[0]
    x = w.strain(0)
    for delays in (np.zeros_like(b.delays), np.full_like(b.delays, 3000), b.delays):
        plan = sp.Plan(b.a1, b.b0, delays, max_block=512, time_chunks=1)
        orc = oracle_mod.FilterOracle(b.a1, b.b0, delays)
        buf = torch.from_numpy(np.concatenate([np.zeros((1, 1), np.float32), x], 1)).cuda()
        zs, rs = [], []
        for i in range(8):
            seg = buf[:, 1 + 512 * i: 1 + 512 * (i + 1)].contiguous() if i % 2 else None
            if seg is None:                     # misaligned view: data_ptr is 4 bytes off a 16-byte boundary
                flat = buf.reshape(-1)[1 + 512 * i: 1 + 512 * (i + 1)]
                assert flat.data_ptr() % 16 != 0
                seg = flat
            zs.append(plan.filter(seg).cpu().numpy())
            rs.append(orc.filter(x[:, 512 * i: 512 * (i + 1)]))
        assert_parity(np.concatenate(zs, -1), np.concatenate(rs, -1), "delays/alignment")


def test_empty_block_reset_and_resume_on_a_fresh_plan(sp, oracle_mod):
    """Resume state = filter state y AND the last d_max inputs.  y is compared element by element with L one-filter
    oracles; a FRESH plan restored from (y, hist) must reproduce block 1 bit-exactly (checkpoint / resume)."""
    import torch
    w = _inputs().config(1, n_templates=9, n_filters=40)
    b = w.banks[0]
    mk = lambda: sp.Plan(b.a1, b.b0, b.delays, max_block=4096, time_chunks=1)
    plan = mk()
    x0, x1 = w.strain(0), w.strain(1)
    empty = torch.empty((1, 0), dtype=torch.float32, device="cuda")
    assert plan.filter(empty).shape == (1, 9, 0)                       # n = 0 is a no-op
    z0 = plan.filter(torch.from_numpy(x0).cuda()).cpu().numpy()
    y, hist = plan.get_state()
    z1 = plan.filter(torch.from_numpy(x1).cuda()).cpu().numpy()
    # y[t][l] is Eq. 7's state after block 0: the last output of the one-filter oracle (t, l)
    assert plan.history_len == int(b.delays.max()) and hist.shape == (1, plan.history_len)
    np.testing.assert_array_equal(hist.cpu().numpy()[0], x0[0, -plan.history_len:])
    yh = y.cpu().numpy()[0]
    for t in range(9):
        ones = oracle_mod.FilterOracle(b.a1[t][:, None], b.b0[t][:, None], b.delays[t][:, None]).filter(x0)[0, :, -1]
        np.testing.assert_allclose(yh[t], ones, rtol=0, atol=2e-5 * np.abs(ones).max())
    plan.reset()
    z0b = plan.filter(torch.from_numpy(x0).cuda()).cpu().numpy()
    np.testing.assert_array_equal(z0, z0b)                              # reset == fresh plan
    fresh = mk()                                                        # never saw x0
    fresh.set_state(y, hist)
    z1b = fresh.filter(torch.from_numpy(x1).cuda()).cpu().numpy()
    np.testing.assert_array_equal(z1, z1b)                              # restored state continues the stream
    wrong = mk()
    wrong.set_state(y, torch.zeros_like(hist))                          # y alone is NOT the resume state
    assert not np.array_equal(wrong.filter(torch.from_numpy(x1).cuda()).cpu().numpy(), z1)
    with pytest.raises(sp.SpiirError) as e:
        plan.filter(torch.zeros((1, 5000), dtype=torch.float32, device="cuda"))
    assert e.value.status == sp.SPIIR_ESTATE
    with pytest.raises(ValueError):
        plan.filter(torch.zeros((1, 64), dtype=torch.float32, device="cuda"), out=torch.zeros(5, dtype=torch.complex64, device="cuda"))


def test_caller_owned_workspace_and_no_hidden_allocation(sp):
    """every device byte of a plan comes from the caller (a torch tensor).  With a workspace the create
    calls of all three plan kinds leave the driver's free memory untouched; a short workspace is refused."""
    import ctypes
    import torch
    L = sp.lib()
    w = _inputs().config(3, n_templates=16)
    b = w.banks[2]
    T, Lf = b.a1.shape
    pool = torch.empty(64 << 20, dtype=torch.uint8, device="cuda")      # everything below is carved from this
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    need = L.spiir_plan_workspace_bytes(T, Lf, int(b.delays.max()), 1, 1024, 0)
    assert 0 < need < pool.numel()
    h = ctypes.c_void_p()
    opts = sp._PlanOpts(1, 1024, 0, 0, pool.data_ptr(), need - 256)
    assert L.spiir_plan_create(ctypes.byref(h), b.a1.ctypes.data, b.b0.ctypes.data, b.delays.ctypes.data, T, Lf, 1024,
                               ctypes.byref(opts)) == sp.SPIIR_ENOMEM
    opts = sp._PlanOpts(1, 1024, 0, 0, pool.data_ptr() + 8, need)
    assert L.spiir_plan_create(ctypes.byref(h), b.a1.ctypes.data, b.b0.ctypes.data, b.delays.ctypes.data, T, Lf, 1024,
                               ctypes.byref(opts)) == sp.SPIIR_EINVAL     # misaligned
    opts = sp._PlanOpts(1, 1024, 0, 0, pool.data_ptr(), need)
    assert L.spiir_plan_create(ctypes.byref(h), b.a1.ctypes.data, b.b0.ctypes.data, b.delays.ctypes.data, T, Lf, 1024,
                               ctypes.byref(opts)) == sp.SPIIR_OK
    x = torch.randn(1, 1024, device="cuda")
    out = torch.empty((1, T, 1024), dtype=torch.complex64, device="cuda")
    assert L.spiir_filter(h, x.data_ptr(), 1024, out.data_ptr(), None) == sp.SPIIR_OK
    off = (need + 255) // 256 * 256
    rn = L.spiir_resamp_workspace_bytes(sp.SPIIR_UP2, 192, 37)
    ropts = sp._ResampOpts(512, pool.data_ptr() + off, rn)
    hr = ctypes.c_void_p()
    assert L.spiir_resamp_create(ctypes.byref(hr), sp.SPIIR_UP2, 192, 5.0, 0.25, 37, ctypes.byref(ropts)) == sp.SPIIR_OK
    off += (rn + 255) // 256 * 256
    H = len(w.banks)
    arrs = [(np.ascontiguousarray(k.a1), np.ascontiguousarray(k.b0), np.ascontiguousarray(k.delays)) for k in w.banks]
    vp = ctypes.c_void_p
    nf = (ctypes.c_int * H)(*[a[0].shape[1] for a in arrs])
    dm = (ctypes.c_int * H)(*[int(a[2].max()) for a in arrs])
    rates = (ctypes.c_int * H)(*[k.rate_hz for k in w.banks])
    mo = sp._MrOpts(1, 4096, 192, 5.0, 0.25, 192, 5.0, 0.25, None, 0)
    mn = L.spiir_mr_workspace_bytes(H, nf, dm, 16, ctypes.byref(mo))
    assert 0 < mn < pool.numel() - off
    mo.workspace, mo.workspace_bytes = pool.data_ptr() + off, mn
    hm = ctypes.c_void_p()
    assert L.spiir_mr_plan_create(ctypes.byref(hm), H, rates, (vp * H)(*[a[0].ctypes.data for a in arrs]),
                                  (vp * H)(*[a[1].ctypes.data for a in arrs]), (vp * H)(*[a[2].ctypes.data for a in arrs]),
                                  nf, 16, ctypes.byref(mo)) == sp.SPIIR_OK
    xm = torch.randn(1, 4096, device="cuda")
    om = torch.empty((1, 16, 4096), dtype=torch.complex64, device="cuda")
    assert L.spiir_mr_filter(hm, xm.data_ptr(), 4096, om.data_ptr(), None) == sp.SPIIR_OK
    torch.cuda.synchronize()
    assert torch.isfinite(torch.view_as_real(om)).all() and torch.isfinite(torch.view_as_real(out)).all()
    # x, out, xm, om came from torch's cached pool or new torch segments; the library itself took nothing:
    # (free memory can only have dropped by what torch allocated for those four tensors, < 4 MiB)
    assert free0 - torch.cuda.mem_get_info()[0] <= (4 << 20)
    L.spiir_mr_plan_destroy(hm); L.spiir_resamp_destroy(hr); L.spiir_plan_destroy(h)
    # the Python classes always pass a torch workspace
    plan = sp.Plan(b.a1, b.b0, b.delays, max_block=256)
    assert plan._ws is not None and plan._ws.numel() == L.spiir_plan_workspace_bytes(T, Lf, int(b.delays.max()), 1, 256, 0)


# ------------------------------------------------------------------------------------------------
# resamplers (exported stages)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("rows,blocks", [(3, (4096, 2, 250, 1024)), (1, (64,) * 5), (70, (2048,))])
def test_resample_down(sp, oracle_mod, rows, blocks):
    import torch
    rng = np.random.default_rng(rows)
    r = sp.Resampler("down", rows, max_block=4096)
    o = oracle_mod.ResampOracle("down", rows)
    zs, rs = [], []
    for n in blocks:
        u = rng.standard_normal((rows, n)).astype(np.float32)
        zs.append(r.down(torch.from_numpy(u).cuda()).cpu().numpy())
        rs.append(o.down(u))
    z, ref = np.concatenate(zs, -1), np.concatenate(rs, -1)
    assert_parity(z.astype(np.complex128), ref.astype(np.complex128), "down2")


@pytest.mark.parametrize("rows,blocks", [(5, (2048, 1, 3, 500)), (2, (32,) * 6), (130, (1024,))])
def test_resample_up_and_accumulate(sp, oracle_mod, rows, blocks):
    import torch
    rng = np.random.default_rng(rows + 100)
    r = sp.Resampler("up", rows, max_block=2048)
    o = oracle_mod.ResampOracle("up", rows)
    zs, rs = [], []
    for i, n in enumerate(blocks):
        v = (rng.standard_normal((rows, n)) + 1j * rng.standard_normal((rows, n))).astype(np.complex64)
        if i % 2 == 0:
            zs.append(r.up(torch.from_numpy(v).cuda()).cpu().numpy())
            rs.append(o.up(v))
        else:                                   # accumulate into an existing base-rate series
            base = (rng.standard_normal((rows, 2 * n)) + 1j * rng.standard_normal((rows, 2 * n))).astype(np.complex64)
            out = torch.from_numpy(base).cuda()
            r.up(torch.from_numpy(v).cuda(), out=out, accumulate=True)
            zs.append(out.cpu().numpy())
            rs.append(o.up(v, out=base.astype(np.complex128)))
    assert_parity(np.concatenate(zs, -1), np.concatenate(rs, -1), "up2")


@pytest.mark.parametrize("n_taps", [192, 32])
@pytest.mark.parametrize("rows,blocks,acc", [(130, (1024, 512, 576), True), (49, (2048, 1400), False), (700, (128, 160, 96), True),
                                             (100, (1001, 777, 40, 1333), True)])    # odd lengths: rows not 16-byte aligned, no TMA staging; a short block
def test_resample_up_tensor_core_path(sp, oracle_mod, rows, blocks, acc, n_taps):
    """The 192-tap (configs[3]) and 32-tap (the paper's own) up stages of a large call run on the tensor cores
    (tcgen05: TF32 product + two bf16 correction products): streamed blocks (history carried through the
    loader), partial strips of rows, partial time tiles, with and without accumulation, against the float64 oracle AND
    against the CUDA-core kernels (flags = 1)."""
    import torch
    rng = np.random.default_rng(rows + n_taps)
    tcr = sp.Resampler("up", rows, max_block=max(blocks), n_taps=n_taps)
    ccr = sp.Resampler("up", rows, max_block=max(blocks), n_taps=n_taps, flags=1)
    orc = oracle_mod.ResampOracle("up", rows, n_taps=n_taps)
    for n in blocks:
        assert rows * n >= 65536 or n == 40                             # the size from which spiir_resample_up goes to the tensor cores
        v = (rng.standard_normal((rows, n)) + 1j * rng.standard_normal((rows, n))).astype(np.complex64)
        base = (rng.standard_normal((rows, 2 * n)) + 1j * rng.standard_normal((rows, 2 * n))).astype(np.complex64)
        o1 = torch.from_numpy(base.copy()).cuda()
        o2 = torch.from_numpy(base.copy()).cuda()
        tcr.up(torch.from_numpy(v).cuda(), o1, accumulate=acc)
        ccr.up(torch.from_numpy(v).cuda(), o2, accumulate=acc)
        ref = orc.up(v) + (base.astype(np.complex128) if acc else 0.0)
        assert_parity(o1.cpu().numpy(), ref, f"tensor-core up taps={n_taps} rows={rows} n={n}")
        assert_parity(o2.cpu().numpy(), ref, f"cuda-core up taps={n_taps} rows={rows} n={n}")


@pytest.mark.parametrize("n_taps", [32, 64, 192, 384])
def test_resamplers_other_tap_counts_and_odd_shapes(sp, oracle_mod, n_taps):
    """32, 192 and (down only) 384 taps take the register-blocked kernels (taps in the kernel parameters), 64 and
    the 384-tap up stage the generic ones; shapes that are not multiples of the per-thread blocking (5 inputs up,
    10 outputs down).  PAPER.md:88: the paper's own filters are 384 taps down and 32 taps up."""
    import torch
    rng = np.random.default_rng(n_taps)
    rows = 37
    rd, ru = sp.Resampler("down", rows, max_block=3000, n_taps=n_taps), sp.Resampler("up", rows, max_block=1500, n_taps=n_taps)
    od, ou = oracle_mod.ResampOracle("down", rows, n_taps=n_taps), oracle_mod.ResampOracle("up", rows, n_taps=n_taps)
    zd, refd, zu, refu = [], [], [], []
    for n in (2, 46, 2998, 1282, 20):
        u = rng.standard_normal((rows, n)).astype(np.float32)
        zd.append(rd.down(torch.from_numpy(u).cuda()).cpu().numpy()); refd.append(od.down(u))
    for n in (1, 7, 1499, 641, 640, 13):
        v = (rng.standard_normal((rows, n)) + 1j * rng.standard_normal((rows, n))).astype(np.complex64)
        base = (rng.standard_normal((rows, 2 * n)) + 1j * rng.standard_normal((rows, 2 * n))).astype(np.complex64)
        out = torch.from_numpy(base).cuda()
        ru.up(torch.from_numpy(v).cuda(), out=out, accumulate=True)
        zu.append(out.cpu().numpy()); refu.append(ou.up(v, out=base.astype(np.complex128)))
    assert_parity(np.concatenate(zd, -1).astype(np.complex128), np.concatenate(refd, -1).astype(np.complex128), f"down2 N={n_taps}")
    assert_parity(np.concatenate(zu, -1), np.concatenate(refu, -1), f"up2 N={n_taps}")


def test_up_stage_short_blocks_many_rows_and_unaligned_input(sp, oracle_mod):
    """(a) rows >= 128 with n_in in {1, 4, 10}: the register-blocked 192-tap kernel packs many rows into a CTA and must
    stay inside its shared-memory limit; (b) a 32-tap stage fed from a complex64 view that starts at an odd element
    (8-byte but not 16-byte aligned): the streaming kernel's 16-byte loads do not apply, the blocked kernel does."""
    import torch
    rng = np.random.default_rng(5)
    rows = 160
    r = sp.Resampler("up", rows, max_block=64)
    o = oracle_mod.ResampOracle("up", rows)
    zs, rs = [], []
    for n in (1, 4, 10, 64, 10, 1):
        v = (rng.standard_normal((rows, n)) + 1j * rng.standard_normal((rows, n))).astype(np.complex64)
        zs.append(r.up(torch.from_numpy(v).cuda()).cpu().numpy()); rs.append(o.up(v))
    assert_parity(np.concatenate(zs, -1), np.concatenate(rs, -1), "up2 many rows, short blocks")
    rows = 6
    r32 = sp.Resampler("up", rows, max_block=256, n_taps=32)
    o32 = oracle_mod.ResampOracle("up", rows, n_taps=32)
    zs, rs = [], []
    for n in (256, 100, 256):
        v = (rng.standard_normal((rows, n)) + 1j * rng.standard_normal((rows, n))).astype(np.complex64)
        buf = torch.zeros(rows * n + 1, dtype=torch.complex64, device="cuda")
        buf[1:] = torch.from_numpy(v).cuda().reshape(-1)
        view = buf[1:].reshape(rows, n)
        assert view.data_ptr() % 16 == 8 and view.is_contiguous()
        zs.append(r32.up(view).cpu().numpy()); rs.append(o32.up(v))
    assert_parity(np.concatenate(zs, -1), np.concatenate(rs, -1), "up2 32 taps, odd-element view")
    with pytest.raises(ValueError):
        r32.up(torch.zeros((rows + 1, 8), dtype=torch.complex64, device="cuda"))          # wrong row count is refused


def test_resampler_state_resume(sp):
    import torch
    rng = np.random.default_rng(9)
    for direction, dt in (("down", np.float32), ("up", np.complex64)):
        mk = lambda: sp.Resampler(direction, 5, max_block=512)
        gen = lambda n: (rng.standard_normal((5, n)) + (1j * rng.standard_normal((5, n)) if direction == "up" else 0)).astype(dt)
        call = lambda r, u: (r.down(torch.from_numpy(u).cuda()) if direction == "down" else r.up(torch.from_numpy(u).cuda())).cpu().numpy()
        r = mk()
        u0, u1 = gen(512), gen(64)
        call(r, u0)
        h = r.get_state()
        assert h.shape == (5, r.history_len) and r.history_len == (191 if direction == "down" else 95)
        np.testing.assert_array_equal(h.cpu().numpy(), u0[:, -r.history_len:])
        z1 = call(r, u1)
        fresh = mk()
        fresh.set_state(h)
        np.testing.assert_array_equal(call(fresh, u1), z1)


def test_multirate_paper_filters_and_state_resume(sp, oracle_mod):
    """a 384-tap (~100 dB) down filter and a 32-tap (~60 dB) up filter in one plan; and the whole
    multirate resume state as one blob restored into a FRESH plan."""
    import torch
    w = _inputs().config(3, n_templates=10)
    banks = [(b.a1, b.b0, b.delays) for b in w.banks]
    kw = dict(n_taps_down=384, kaiser_beta_down=10.0, n_taps_up=32, kaiser_beta_up=5.0)
    mk = lambda: sp.MultiratePlan(banks, [b.rate_hz for b in w.banks], max_block=1024, **kw)
    plan = mk()
    assert plan.launches(1024) <= 1 + 1 + 7 + 3          # fused 384-tap down chain, fused 32-tap up cascade, banks
    orc = oracle_mod.MultirateOracle(banks, n_taps_down=384, beta_down=10.0, n_taps_up=32, beta_up=5.0)
    rng = np.random.default_rng(384)
    xs = [rng.standard_normal((1, n)).astype(np.float32) for n in (1024, 64, 448)]
    z = stream_gpu_plan(plan, xs)
    assert_parity(z, stream_oracle(orc, xs), "multirate 384 down / 32 up")
    blob = plan.get_state()
    x3 = rng.standard_normal((1, 512)).astype(np.float32)
    z3 = plan.filter(torch.from_numpy(x3).cuda()).cpu().numpy()
    assert_parity(z3, orc.filter(x3), "multirate 384 down / 32 up, block 4")
    fresh = mk()
    fresh.set_state(blob)
    np.testing.assert_array_equal(fresh.filter(torch.from_numpy(x3).cuda()).cpu().numpy(), z3)


@pytest.mark.parametrize("T,L", [(6, 256), (3, 513), (40, 5), (9, 32), (5, 100)])
def test_paper_design_comparison_kernels(sp, oracle_mod, T, L):
    """The paper's own mapping (thread per filter, __ldg, warp shuffle, atomicAdd DA) computes the same
    SNR; float atomics make the order of the cross-warp sum free, so parity is by tolerance only (F8)."""
    w = _inputs().config(0, n_templates=T, n_filters=L)
    b = w.banks[0]
    pd = sp.PaperDesignPlan(b.a1, b.b0, b.delays, max_block=800)
    rng = np.random.default_rng(L)
    xs = [rng.standard_normal((1, n)).astype(np.float32) for n in (800, 100, 37)]
    z = stream_gpu_plan(pd, xs)
    ref = stream_oracle(oracle_mod.FilterOracle(b.a1, b.b0, b.delays), xs)
    assert_parity(z, ref, f"paper design T={T} L={L}")


@pytest.mark.parametrize("n_taps,blocks", [(192, (192, 64, 448)), (32, (256, 128)), (64, (256, 64))])
def test_multirate_fused_chains_and_fallback(sp, oracle_mod, n_taps, blocks):
    """192 taps: fused down chain + fused up cascade; 32 taps: fused up cascade, per-stage down kernels;
    64 taps: one launch per stage both ways.  Ragged block lengths (multiples of 2^(H-1) only)."""
    w = _inputs().config(3, n_templates=9)
    banks = [(b.a1, b.b0, b.delays) for b in w.banks]
    plan = sp.MultiratePlan(banks, [b.rate_hz for b in w.banks], max_block=512, n_taps=n_taps)
    orc = oracle_mod.MultirateOracle(banks, n_taps=n_taps)
    rng = np.random.default_rng(n_taps + 1)
    xs = [rng.standard_normal((1, n)).astype(np.float32) for n in blocks]
    z = stream_gpu_plan(plan, xs)
    ref = stream_oracle(orc, xs)
    assert_parity(z, ref, f"multirate N={n_taps}")
    expect = {192: 2, 32: 1 + 6, 64: 12}[n_taps]
    assert plan.launches(256) >= expect


def test_multirate_two_streams(sp, oracle_mod):
    """Two independent strain streams through the fused down chain (one CTA per stream) and the fused
    up cascade (one CTA per (stream, template) row)."""
    w = _inputs().config(3, n_templates=7)
    banks = [(b.a1, b.b0, b.delays) for b in w.banks]
    plan = sp.MultiratePlan(banks, [b.rate_hz for b in w.banks], n_streams=2, max_block=512)
    orc = oracle_mod.MultirateOracle(banks, n_streams=2)
    rng = np.random.default_rng(77)
    xs = [rng.standard_normal((2, n)).astype(np.float32) for n in (320, 64, 512)]
    z = stream_gpu_plan(plan, xs)
    ref = stream_oracle(orc, xs)
    assert z.shape == (2, 7, 896)
    assert_parity(z, ref, "multirate S=2")
    # the two streams are independent: stream 1 alone gives the same series
    plan1 = sp.MultiratePlan(banks, [b.rate_hz for b in w.banks], n_streams=1, max_block=512)
    z1 = stream_gpu_plan(plan1, [x[1:2] for x in xs])
    np.testing.assert_array_equal(z1[0], z[1])


def test_multirate_long_block_falls_back_to_per_stage_launches(sp, oracle_mod):
    """A block too long for the fused chains' shared-memory buffers: one launch per stage instead
    (and the banks tile their windows in time)."""
    inp = _inputs()
    rates = [4096, 2048, 1024]
    banks = []
    for h, (R, L) in enumerate(zip(rates, (6, 20, 40))):
        b = inp.make_bank((9, 9, h), 3, L, R, 0.9, 0.9999, 300)
        banks.append((b.a1, b.b0, b.delays))
    n = 65536
    plan = sp.MultiratePlan(banks, rates, max_block=n)
    # 65536 samples: 2 + 2 per-stage resampling launches (the fused chains would need > 227 KB) + >= 1 per bank
    assert plan.launches(n) >= 4 + 3
    orc = oracle_mod.MultirateOracle(banks)
    rng = np.random.default_rng(3)
    xs = [rng.standard_normal((1, m)).astype(np.float32) for m in (n, 4096)]
    z = stream_gpu_plan(plan, xs)
    ref = stream_oracle(orc, xs)
    assert_parity(z, ref, "multirate long block")


def test_kaiser_taps_match_oracle_design(sp, oracle_mod):
    """The library generates its own taps (no shared table); they agree with the oracle's to 1 ulp."""
    h = sp.spiir_kaiser_taps(192, 5.0, 0.25)
    _, h32 = oracle_mod.kaiser_taps(192, 5.0, 0.25)
    assert np.max(np.abs(h.astype(np.float64) - h32.astype(np.float64)) / np.spacing(np.abs(h32)).astype(np.float64)) <= 1.0


# ------------------------------------------------------------------------------------------------
# the configs at their FULL sizes and FULL block counts, in the launch geometry bench.py times:
# configs[1] and configs[3] against the oracle on the WHOLE bank; configs[4] on >= 256 templates per stream that
# touch every persistent CTA (CTA bx of a stream owns templates bx*8 + j*1184 .. +8) and include the first and last;
# configs[2] sweep points on sampled templates.  Errors are accumulated block by block over the whole run (F10).
# ------------------------------------------------------------------------------------------------
def _cfg4_templates():
    idx = {0, 1, 7, 8, 16383, 16382, 8191, 8192}
    idx |= {bx * 8 + (bx % 8) + 1184 * (bx % 13) for bx in range(148)}
    idx |= set(range(5, 16384, 151))
    idx = np.array(sorted(i for i in idx if i < 16384))
    assert idx.size >= 256 and len({(i % 1184) // 8 for i in idx.tolist()}) == 148
    return idx


@pytest.mark.parametrize("cfg,kw,nblk,idx", [
    (1, {}, 16, None),
    (2, {"n_filters": 1}, 64, [0, 17, 2048, 4095]),
    (2, {"n_filters": 4}, 64, [0, 17, 2048, 4095]),
    (2, {"n_filters": 32}, 64, [0, 17, 2048, 4095]),
    (3, {}, 32, None),
    (4, {}, 64, "cfg4"),
])
def test_full_size_full_length_streams(sp, oracle_mod, cfg, kw, nblk, idx):
    import torch
    w = _inputs().config(cfg, **kw)
    idx = _cfg4_templates() if isinstance(idx, str) else (np.arange(w.n_templates) if idx is None else np.array(idx))
    if len(w.banks) == 1:
        b = w.banks[0]
        plan = sp.Plan(b.a1, b.b0, b.delays, b.rate_hz, n_streams=w.n_streams, max_block=w.block)
        orc = oracle_mod.FilterOracle(b.a1[idx], b.b0[idx], b.delays[idx], w.n_streams)
    else:
        banks = [(b.a1, b.b0, b.delays) for b in w.banks]
        plan = sp.MultiratePlan(banks, [b.rate_hz for b in w.banks], n_streams=w.n_streams, max_block=w.block)
        orc = oracle_mod.MultirateOracle([(a[idx], b0[idx], d[idx]) for a, b0, d in banks], w.n_streams)
    assert nblk == w.n_blocks
    out = torch.empty((w.n_streams, w.n_templates, w.block), dtype=torch.complex64, device="cuda")
    didx = torch.from_numpy(idx).cuda()
    acc = ParityAccumulator()
    for i in range(nblk):
        x = w.strain(i)
        plan.filter(torch.from_numpy(x).cuda(), out)
        z = out.cpu().numpy() if idx.size == w.n_templates else out[:, didx].cpu().numpy()
        acc.add(z, orc.filter(x))
    rel, mab = acc.check(f"{w.name} full length, {idx.size} templates")
    print(f"{w.name}: {idx.size} templates x {nblk} blocks  rel-L2 {rel:.2e}  max-abs ratio {mab:.2e}")


# ------------------------------------------------------------------------------------------------
# CUDA graphs: the ping-pong phase of every carried history lives on the device, so one captured
# call can be replayed for every block of a stream
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kind", ["few_filter_chunked", "many_filter", "multirate"])
def test_cuda_graph_replay_continues_the_stream(sp, oracle_mod, kind):
    import torch
    inp = _inputs()
    if kind == "multirate":
        w = inp.config(3, n_templates=12, n_blocks=5)
        banks = [(b.a1, b.b0, b.delays) for b in w.banks]
        plan = sp.MultiratePlan(banks, [b.rate_hz for b in w.banks], max_block=w.block)
        orc = oracle_mod.MultirateOracle(banks)
        T = 12
    else:
        w = inp.config(2, n_templates=300, n_filters=8, n_blocks=5) if kind == "few_filter_chunked" else \
            inp.config(1, n_templates=20, n_blocks=5)
        b = w.banks[0]
        plan = sp.Plan(b.a1, b.b0, b.delays, b.rate_hz, max_block=w.block)
        orc = oracle_mod.FilterOracle(b.a1, b.b0, b.delays)
        T = b.a1.shape[0]
    xs = [w.strain(i) for i in range(5)]
    x_static = torch.zeros((1, w.block), dtype=torch.float32, device="cuda")
    out_static = torch.zeros((1, T, w.block), dtype=torch.complex64, device="cuda")
    # warm-up outside the capture (sets kernel attributes), then start the stream again
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        plan.filter(x_static, out_static)
    torch.cuda.current_stream().wait_stream(side)
    plan.reset()
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        plan.filter(x_static, out_static)
    plan.reset()                      # whatever the capture did to host-side bookkeeping, the device state restarts
    outs = []
    for x in xs:
        x_static.copy_(torch.from_numpy(x))
        g.replay()
        outs.append(out_static.cpu().numpy().copy())
    z = np.concatenate(outs, -1)
    ref = stream_oracle(orc, xs)
    assert_parity(z, ref, f"graph replay {kind}")
