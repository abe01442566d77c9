"""GPU parity: the CUDA path (through the C ABI) against the float64 oracle, element by element,
on the same seeded inputs.  Tolerances are BASELINE.json north_star's (tests/_util.py).

Sizes: cut-down configs the oracle finishes in seconds (several tiles, ragged tails), plus the
full BASELINE.json sizes in the launch configuration bench.py times, checked on sampled templates
the oracle computes one by one (every template is an independent unit).
"""
import numpy as np
import pytest

from _util import assert_parity, stream_gpu_plan, stream_oracle

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
    """Banks of 32..128 filters with >= 2368 templates put two templates in a warp (16 lanes each)."""
    for L in (40, 128):
        w = _inputs().config(1, n_templates=2400, n_filters=L)
        b = w.banks[0]
        plan = sp.Plan(b.a1, b.b0, b.delays % 300, b.rate_hz, max_block=256)
        info = plan.launch_info(256)
        assert info["lanes_per_template"] == 16 and info["F"] == (L + 15) // 16
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


def test_unsupported_filter_count(sp):
    w = _inputs().config(0, n_templates=1, n_filters=513)
    b = w.banks[0]
    with pytest.raises(sp.SpiirError) as e:
        sp.Plan(b.a1, b.b0, b.delays)
    assert e.value.status == sp.SPIIR_EUNSUPPORTED


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


def test_empty_block_reset_and_state_roundtrip(sp, oracle_mod):
    import torch
    w = _inputs().config(1, n_templates=9)
    b = w.banks[0]
    plan = sp.Plan(b.a1, b.b0, b.delays, max_block=4096, time_chunks=1)
    x0, x1 = w.strain(0), w.strain(1)
    empty = torch.empty((1, 0), dtype=torch.float32, device="cuda")
    assert plan.filter(empty).shape == (1, 9, 0)                       # n = 0 is a no-op
    z0 = plan.filter(torch.from_numpy(x0).cuda()).cpu().numpy()
    y = plan.get_state()
    z1 = plan.filter(torch.from_numpy(x1).cuda()).cpu().numpy()
    # the carried state is Eq. 7's y after block 0, in the caller's [S][T][L] order
    orc = oracle_mod.FilterOracle(b.a1, b.b0, b.delays)
    orc.filter(x0)
    # one-filter-at-a-time check of the state through the closed form: state sums to z0's last sample
    np.testing.assert_allclose(y.cpu().numpy().sum(-1)[0], z0[0, :, -1], rtol=2e-4, atol=1e-7)
    plan.reset()
    z0b = plan.filter(torch.from_numpy(x0).cuda()).cpu().numpy()
    np.testing.assert_array_equal(z0, z0b)                              # reset == fresh plan
    plan.set_state(y)
    z1b = plan.filter(torch.from_numpy(x1).cuda()).cpu().numpy()
    np.testing.assert_array_equal(z1, z1b)                              # restored state continues the stream
    with pytest.raises(sp.SpiirError) as e:
        plan.filter(torch.zeros((1, 5000), dtype=torch.float32, device="cuda"))
    assert e.value.status == sp.SPIIR_ESTATE


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


@pytest.mark.parametrize("n_taps", [32, 64, 192])
def test_resamplers_other_tap_counts_and_odd_shapes(sp, oracle_mod, n_taps):
    """32 and 192 taps take the register-blocked kernels (taps in the kernel parameters), 64 the generic
    ones; shapes that are not multiples of the per-thread blocking (5 inputs up, 10 outputs down)."""
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
# the five configs at their FULL sizes and FULL block counts, oracle on sampled templates
# (templates are independent units; the tolerance is over the whole run, reading F10)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,kw,nblk,idx", [
    (1, {}, 16, [0, 1, 7, 500, 1023]),
    (2, {"n_filters": 1}, 64, [0, 17, 2048, 4095]),
    (2, {"n_filters": 4}, 64, [0, 17, 2048, 4095]),
    (2, {"n_filters": 32}, 64, [0, 17, 2048, 4095]),
    (3, {}, 32, [0, 511, 1023]),
    (4, {}, 64, [0, 8191, 16383]),
])
def test_full_size_full_length_streams_sampled(sp, oracle_mod, cfg, kw, nblk, idx):
    import torch
    w = _inputs().config(cfg, **kw)
    idx = np.array(idx)
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
    zs, refs = [], []
    for i in range(nblk):
        x = w.strain(i)
        plan.filter(torch.from_numpy(x).cuda(), out)
        zs.append(out[:, idx].cpu().numpy())
        refs.append(orc.filter(x))
    assert_parity(np.concatenate(zs, -1), np.concatenate(refs, -1), f"{w.name} full length")


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
