"""spiir_filter_block_noalloc (include/spiir.h, "NO-ALLOCATION ENTRY POINT"): the entry point whose scan scratch is a
device array built into the library, against the existing plan-based path (spiir_plan_create + spiir_filter on a fresh
plan) on the same seeded inputs, within the parity tolerance of every other GPU test (tests/_util.py), on two calls in
a row that share the array.  The file name sorts last so that `pytest -x` reaches it after every other test.
"""
import ctypes

import numpy as np
import pytest

from _util import assert_parity


@pytest.fixture(scope="module")
def sp():
    import paper_1702_02256_b200 as sp
    sp.lib()                       # fails loudly when the extension is missing
    return sp


def _case(index, T, L, n, seed):
    """(bank, x): a cut of BASELINE.json configs[index] (same distributions) and one block of unit-variance noise."""
    from paper_1702_02256_b200 import inputs
    w = inputs.config(index, n_templates=T, n_filters=L)
    x = np.random.default_rng(seed).standard_normal(n).astype(np.float32)
    return w.banks[0], x


def _existing_path(sp, bank, x):
    import torch
    plan = sp.Plan(bank.a1, bank.b0, bank.delays, bank.rate_hz, max_block=len(x))
    z = plan.filter(torch.from_numpy(x).cuda()).cpu().numpy()[0]
    plan.close()
    return z


def _device_args(bank, x):
    import torch
    return tuple(torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (bank.a1, bank.b0, bank.delays, x))


def _noalloc(sp, bank, x, out=None, time_chunks=0):
    import torch
    z = sp.filter_block_noalloc(*_device_args(bank, x), out=out, time_chunks=time_chunks)
    torch.cuda.synchronize()
    return z.cpu().numpy()


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_plan_path(sp):
    import torch
    # call 1: 16 templates x 128 filters, 4096 samples (configs[0]): 64 chunks, 1 MiB of the array
    bank1, x1 = _case(0, 16, 128, 4096, 11)
    # call 2: another shape and other data over the same array: 37 x 20 filters, ragged 1500 samples, 23 chunks
    bank2, x2 = _case(2, 37, 20, 1500, 12)
    assert sp.noalloc_scratch_need(16, 128, 4096) == 64 * 16 * 128 * 8
    sp.noalloc_setup()
    args1, args2 = _device_args(bank1, x1), _device_args(bank2, x2)
    out1 = torch.empty((16, 4096), dtype=torch.complex64, device="cuda")
    out2 = torch.empty((37, 1500), dtype=torch.complex64, device="cuda")
    sp.filter_block_noalloc(*args2, out=out2)                # warm-up: the kernels' module is loaded before the free-memory reading
    torch.cuda.synchronize()
    out2.zero_()
    free_before = torch.cuda.mem_get_info()[0]
    sp.filter_block_noalloc(*args1, out=out1)                # two calls in a row on one stream, no synchronisation between
    sp.filter_block_noalloc(*args2, out=out2)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before       # the library took no device memory for them
    z1, z2 = out1.cpu().numpy(), out2.cpu().numpy()
    assert_parity(z1[None], _existing_path(sp, bank1, x1)[None], "no-alloc call 1 vs plan path")
    assert_parity(z2[None], _existing_path(sp, bank2, x2)[None], "no-alloc call 2 vs plan path")
    # the array now holds call 2's chunk states: call 1 again must give call 1's result bit for bit
    assert np.array_equal(_noalloc(sp, bank1, x1), z1)
    # explicit chunk counts (1 = no scan at all, 5 = ragged last chunk) agree too
    for tc in (1, 5):
        assert_parity(_noalloc(sp, bank2, x2, time_chunks=tc)[None], z2[None], f"time_chunks={tc}")


@pytest.mark.gpu
def test_against_the_oracle(sp):
    import oracle
    bank, x = _case(0, 5, 96, 1000, 13)
    ref = oracle.FilterOracle(bank.a1, bank.b0, bank.delays).filter(x[None])[0]
    assert_parity(_noalloc(sp, bank, x)[None], ref[None], "no-alloc vs oracle")


def test_sizes_beyond_the_built_in_array_are_rejected(sp):
    """Size checks come before any CUDA call and before any pointer is touched: runs without a GPU."""
    L = sp.lib()
    limit = sp.SPIIR_NOALLOC_SCRATCH_BYTES
    assert limit == 4 << 20
    dummy = ctypes.c_void_p(256)
    call = lambda T, F, n, tc: L.spiir_filter_block_noalloc(dummy, dummy, dummy, T, F, dummy, n, tc, dummy, None)
    # 2048 x 512 filters = 8 MiB for a single chunk
    assert sp.noalloc_scratch_need(2048, 512, 4096) > limit
    assert call(2048, 512, 4096, 0) == sp.SPIIR_EINVAL
    assert b"scratch" in L.spiir_last_error()
    # fits with 64 chunks, not with 65
    assert sp.noalloc_scratch_need(64, 128, 8192, 64) == limit
    assert call(64, 128, 8192, 65) == sp.SPIIR_EINVAL
    assert call(4, 513, 256, 0) == sp.SPIIR_EUNSUPPORTED
    assert call(0, 8, 256, 0) == sp.SPIIR_EINVAL
