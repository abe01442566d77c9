"""Randomised parity run: seeded random shapes through every entry point of the C ABI against the float64 oracle.

The hand-picked cases of test_gpu_parity.py cover the mappings one by one; this file covers their COMBINATIONS (template
count x filters x streams x delays x block lengths x chunking) -- the phase-word race fixed in spiir_filter.cuh was found
by a longer run of exactly this generator.  Seeds are fixed, so a failure reproduces.
"""
import numpy as np
import pytest

from _util import REL_L2_TOL, MAX_ABS_TOL, parity_errors

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sp():
    import paper_1702_02256_b200 as sp
    sp.lib()
    return sp


def _bank(rng, T, L, dmax):
    mag, arg = rng.uniform(0.5, 0.9999, (T, L)), rng.uniform(0, 2 * np.pi, (T, L))
    a1 = (mag * np.exp(1j * arg)).astype(np.complex64)
    b0 = (1e-3 * (rng.standard_normal((T, L)) + 1j * rng.standard_normal((T, L)))).astype(np.complex64)
    return a1, b0, rng.integers(0, dmax + 1, (T, L)).astype(np.int32)


def _check(z, ref, desc):
    rel, mab = parity_errors(z, ref)
    assert rel <= REL_L2_TOL and mab <= MAX_ABS_TOL, f"{desc}: rel-L2 {rel:.3e}, max-abs ratio {mab:.3e}"


def _cuda(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("seed", [11, 12, 13])
def test_single_rate_plans(sp, seed):
    import oracle
    rng = np.random.default_rng(seed)
    for case in range(40):
        L = int(rng.choice([1, 2, 3, 4, 5, 7, 8, 9, 13, 16, 17, 24, 31, 32, 33, 40, 48, 57, 64, 65, 96, 128, 129, 200, 256, 300, 512, 513, 700]))
        T = int(rng.choice([1, 2, 7, 8, 9, 31, 33, 64, 100, 148, 300, 600, 1030, 2368, 2500])) if L <= 64 else int(rng.choice([1, 3, 8, 20, 64, 150]))
        S = int(rng.choice([1, 1, 2, 3]))
        dmax = int(rng.choice([0, 3, 100, 1000, 3000]))
        maxb = int(rng.choice([16, 100, 256, 1000, 2048, 5000]))
        blocks = [int(rng.integers(1, maxb + 1)) for _ in range(int(rng.integers(1, 4)))]
        tc = int(rng.choice([0, 0, 0, 1, 3]))
        a1, b0, d = _bank(rng, T, L, dmax)
        plan = sp.Plan(a1, b0, d, 4096, n_streams=S, max_block=maxb, time_chunks=tc)
        orc = oracle.FilterOracle(a1, b0, d, S)
        zs, rs = [], []
        for n in blocks:
            x = rng.standard_normal((S, n)).astype(np.float32)
            zs.append(plan.filter(_cuda(x)).cpu().numpy())
            rs.append(orc.filter(x))
        desc = f"seed {seed} case {case}: T={T} L={L} S={S} dmax={dmax} blocks={blocks} time_chunks={tc} {plan.launch_info(maxb)}"
        plan.close()
        _check(np.concatenate(zs, -1), np.concatenate(rs, -1), desc)


@pytest.mark.parametrize("seed", [21, 22])
def test_resume_on_a_fresh_plan(sp, seed):
    import oracle
    rng = np.random.default_rng(seed)
    for case in range(15):
        L = int(rng.choice([1, 4, 24, 32, 64, 256])); T = int(rng.choice([2, 9, 64, 300])); S = int(rng.choice([1, 2]))
        dmax = int(rng.choice([0, 100, 1500])); maxb = int(rng.choice([64, 500, 2048]))
        a1, b0, d = _bank(rng, T, L, dmax)
        n1, n2 = int(rng.integers(1, maxb + 1)), int(rng.integers(1, maxb + 1))
        x1, x2 = rng.standard_normal((S, n1)).astype(np.float32), rng.standard_normal((S, n2)).astype(np.float32)
        p1 = sp.Plan(a1, b0, d, 4096, n_streams=S, max_block=maxb)
        p1.filter(_cuda(x1))
        y, hist = p1.get_state()
        p1.close()
        p2 = sp.Plan(a1, b0, d, 4096, n_streams=S, max_block=maxb, time_chunks=int(rng.choice([0, 1])))
        p2.set_state(y, hist)
        z = p2.filter(_cuda(x2)).cpu().numpy()
        p2.close()
        orc = oracle.FilterOracle(a1, b0, d, S)
        orc.filter(x1)
        _check(z, orc.filter(x2), f"seed {seed} case {case}: resume T={T} L={L} S={S} dmax={dmax} n1={n1} n2={n2}")


@pytest.mark.parametrize("seed", [31, 32])
def test_resamplers(sp, seed):
    import oracle
    import torch
    rng = np.random.default_rng(seed)
    for case in range(24):
        up = bool(rng.integers(0, 2))
        taps = int(rng.choice([32, 192, 64] if up else [32, 192, 384, 64]))
        rows = int(rng.choice([1, 5, 48, 49, 100, 333, 1000] if up else [1, 2, 5, 100, 1000]))
        maxb = int(rng.choice([50, 200, 700, 1500, 3000]))
        nb = int(rng.integers(1, 4))
        acc = bool(rng.integers(0, 2))
        r = sp.Resampler("up" if up else "down", rows, max_block=maxb, n_taps=taps)
        orc = oracle.ResampOracle("up" if up else "down", rows, n_taps=taps)
        zs, rs, blocks = [], [], []
        for _ in range(nb):
            if up:
                n = int(rng.integers(1, maxb + 1))
                v = (rng.standard_normal((rows, n)) + 1j * rng.standard_normal((rows, n))).astype(np.complex64)
                base = (rng.standard_normal((rows, 2 * n)) + 1j * rng.standard_normal((rows, 2 * n))).astype(np.complex64)
                out = torch.from_numpy(base.copy()).cuda()
                r.up(_cuda(v), out, accumulate=acc)
                zs.append(out.cpu().numpy())
                rs.append(orc.up(v) + (base.astype(np.complex128) if acc else 0.0))
            else:
                n = 2 * int(rng.integers(1, maxb // 2 + 1))
                u = rng.standard_normal((rows, n)).astype(np.float32)
                zs.append(r.down(_cuda(u)).cpu().numpy().astype(np.complex128))
                rs.append(orc.down(u).astype(np.complex128))
            blocks.append(n)
        r.close()
        _check(np.concatenate(zs, -1)[None], np.concatenate(rs, -1)[None],
               f"seed {seed} case {case}: {'up' if up else 'down'} taps={taps} rows={rows} blocks={blocks} accumulate={acc}")


@pytest.mark.parametrize("seed", [41])
def test_multirate_plans(sp, seed):
    import oracle
    rng = np.random.default_rng(seed)
    for case in range(12):
        H = int(rng.integers(2, 5)); T = int(rng.choice([1, 3, 8, 40, 130])); S = int(rng.choice([1, 1, 2]))
        rates = [4096 >> h for h in range(H)]
        Ls = [int(rng.choice([1, 4, 8, 16, 24, 32, 48, 64, 100])) for _ in range(H)]
        unit = 1 << (H - 1)
        maxb = unit * int(rng.choice([8, 32, 100, 256]))
        blocks = [unit * int(rng.integers(1, maxb // unit + 1)) for _ in range(int(rng.integers(1, 4)))]
        kw = dict(n_taps_down=384, n_taps_up=32) if rng.integers(0, 3) == 0 else {}
        banks = [_bank(rng, T, Ls[h], int(rng.choice([0, 10, rates[h] // 8]))) for h in range(H)]
        plan = sp.MultiratePlan(banks, rates, n_streams=S, max_block=maxb, **kw)
        orc = oracle.MultirateOracle(banks, n_streams=S, **kw)
        zs, rs = [], []
        for n in blocks:
            x = rng.standard_normal((S, n)).astype(np.float32)
            zs.append(plan.filter(_cuda(x)).cpu().numpy())
            rs.append(orc.filter(x))
        plan.close()
        _check(np.concatenate(zs, -1), np.concatenate(rs, -1), f"seed {seed} case {case}: multirate H={H} T={T} S={S} L={Ls} blocks={blocks} {kw}")
