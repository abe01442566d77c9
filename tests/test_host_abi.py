"""CPU-side checks of the CUDA library: it builds, loads, exports every symbol include/spiir.h
declares, rejects bad arguments without a GPU, and its host logic (filter permutation, launch
geometry, Kaiser taps) behaves as DESIGN.md says.  No compute call is made here."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def sp():
    from paper_1702_02256_b200 import build
    build.build()
    import paper_1702_02256_b200 as sp
    sp.lib()
    return sp


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "spiir.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(spiir_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(sp):
    names = _declared_symbols()
    assert len(names) >= 20
    L = sp.lib()
    for n in names:
        assert hasattr(L, n), f"{n} declared in include/spiir.h but not exported by libspiir.so"
    assert set(sp.EXPORTS) == set(names)
    assert sp.version().startswith("spiir-b200") and "sm_100a" in sp.version()


def test_library_has_sm100a_code_and_packed_fp32(sp):
    """The shipped binary is sm_100a SASS with FFMA2 (packed FP32) and a TMA bulk copy (UBLKCP)."""
    import shutil
    import subprocess
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    out = subprocess.run([cuobjdump, "-sass", sp.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    assert "FFMA2" in out and "UBLKCP" in out and "SYNCS" in out


def test_argument_errors_need_no_gpu(sp):
    L = sp.lib()
    h = ctypes.c_void_p()
    assert L.spiir_plan_create(ctypes.byref(h), None, None, None, 1, 1, 4096, None) == sp.SPIIR_EINVAL
    assert b"NULL" in L.spiir_last_error()
    a = np.zeros((1, 4), np.complex64)
    d = np.array([[0, 1, -1, 2]], np.int32)
    assert L.spiir_plan_create(ctypes.byref(h), a.ctypes.data, a.ctypes.data, d.ctypes.data, 1, 4, 4096, None) == sp.SPIIR_EINVAL
    assert L.spiir_filter(None, None, 16, None, None) == sp.SPIIR_EINVAL
    assert L.spiir_resamp_create(ctypes.byref(h), 0, 191, 5.0, 0.25, 1, None) == sp.SPIIR_EINVAL   # odd tap count
    assert L.spiir_resample_down(None, None, 2, None, None) == sp.SPIIR_EINVAL
    rates = (ctypes.c_int * 2)(4096, 1024)
    assert L.spiir_mr_plan_create(ctypes.byref(h), 2, rates, ctypes.byref(h), ctypes.byref(h), ctypes.byref(h),
                                  rates, 1, None) == sp.SPIIR_EINVAL                                 # rates do not halve


def test_no_gpu_means_create_fails_loudly(sp):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    a = np.full((2, 8), 0.5 + 0.1j, np.complex64)
    d = np.zeros((2, 8), np.int32)
    with pytest.raises(sp.SpiirError) as e:
        sp.Plan(a, a, d)
    assert e.value.status in (sp.SPIIR_ECUDA, sp.SPIIR_ENOMEM)


@pytest.mark.parametrize("L,F,LPT", [(1, 1, 1), (4, 4, 1), (5, 3, 2), (8, 4, 2), (16, 4, 4), (31, 4, 8), (32, 1, 32),
                                      (128, 4, 32), (256, 8, 32), (257, 10, 32), (512, 16, 32)])
def test_lane_mapping(sp, L, F, LPT):
    g = sp.spiir_host_geometry(64, L, 1, 100, 1024)
    assert (g["F"], g["lanes_per_template"]) == (F, LPT)
    assert F * LPT >= L


@pytest.mark.parametrize("L,F,NP", [(513, 6, 3), (544, 6, 3), (600, 5, 4), (1024, 8, 4), (1025, 7, 5), (2048, 8, 8)])
def test_lane_mapping_multi_warp_templates(sp, L, F, NP):
    """a 513-filter template takes 544 threads of one block; here it spans NP warps of one CTA with
    F filters per lane, the pair with the least padding."""
    m = sp.spiir_host_lane_mapping(L)
    assert (m["F"], m["lanes_per_template"], m["warps_per_template"]) == (F, 32, NP)
    assert F * 32 * NP >= L and F <= 8
    g = sp.spiir_host_geometry(64, L, 1, 100, 1024)
    assert g["warps_per_cta"] % NP == 0 and g["warps_per_cta"] <= 8
    with pytest.raises(sp.SpiirError):
        sp.spiir_host_lane_mapping(2049)
    with pytest.raises(sp.SpiirError):
        sp.spiir_host_geometry(4, 2049, 1, 10, 256)


def test_rate_assignment_reading_r8(sp):
    """PAPER.md:79 / DESIGN.md reading R8: lowest available rate whose Nyquist band holds f0 + band_factor * df."""
    rates = [4096, 2048, 1024, 512, 256, 128, 64]
    # |a1| close to 1: negligible bandwidth term; centre frequencies just below / above each rate's Nyquist frequency
    f0 = np.array([10.0, 31.9, 32.1, 63.0, 65.0, 500.0, 513.0, 1023.0, 1025.0, 2047.0])
    a1 = (0.99999 * np.exp(2j * np.pi * f0 / 4096)).astype(np.complex64)          # df = 0.0065 Hz
    idx = sp.spiir_assign_rates(a1, 4096, rates, band_factor=1.0)
    want = [6, 6, 5, 5, 4, 2, 1, 1, 0, 0]
    assert idx.tolist() == want
    # negative frequencies count by magnitude; a strongly damped filter is wide and moves up
    a = np.array([0.999 * np.exp(-2j * np.pi * 100 / 4096), 0.5 * np.exp(2j * np.pi * 100 / 4096)], np.complex64)
    i2 = sp.spiir_assign_rates(a, 4096, rates, band_factor=1.0)
    assert i2[0] == 4 and i2[1] < i2[0]
    assert sp.spiir_assign_rates(a, 4096, rates, band_factor=0.0).tolist() == [4, 4]
    with pytest.raises(sp.SpiirError):
        sp.spiir_assign_rates(a, 4096, [2048, 1024])          # rates[0] must be the base rate


def test_workspace_queries_fail_loudly_without_a_device(sp):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    assert sp.lib().spiir_plan_workspace_bytes(16, 128, 2047, 1, 4096, 0) == 0
    assert b"CUDA" in sp.lib().spiir_last_error()
    assert sp.lib().spiir_resamp_workspace_bytes(0, 192, 3) > 0          # stage sizes need no device
    assert sp.lib().spiir_resamp_workspace_bytes(0, 191, 3) == 0


def test_chunking_follows_the_cost_model(sp):
    # configs[2]: 4096 templates x 1..32 filters, 256-sample blocks -> two more launches never pay; up to 16 filters
    # (several templates per warp) the chunks are the warps of one CTA: still ONE launch
    for L in (1, 2, 4, 8, 16, 32):
        g = sp.spiir_host_geometry(4096, L, 1, 255, 256)
        assert g["launches"] == 1, L
        assert (g["time_chunks"] > 1) == (L <= 16), (L, g)
        assert g["time_chunks"] == 1 or g["warps_per_cta"] == g["time_chunks"]
    assert sp.spiir_host_geometry(4096, 4, 1, 255, 256, time_chunks=1)["time_chunks"] == 1
    # one bulk call of 16384 samples: equal time tiles that fit the shared-memory window
    g = sp.spiir_host_geometry(4096, 1, 1, 255, 16384)
    assert g["launches"] == 1 and g["time_tile"] == 8192 and g["time_chunks"] == 16
    # the two highest rates of configs[3]: 1024 templates x 8 / 16 filters, 4096 / 2048 samples -> scanned inside a CTA
    for L, n in ((8, 4096), (16, 2048)):
        g = sp.spiir_host_geometry(1024, L, 1, n - 1, n)
        assert g["time_chunks"] > 1 and g["launches"] == 1, (L, g)
    # ... but not its lower rates (one warp per template already gives 1024 warps)
    assert sp.spiir_host_geometry(1024, 32, 1, 1023, 1024)["time_chunks"] == 1
    # a long block of a small bank is chunked, a short one is not
    assert sp.spiir_host_geometry(16, 128, 1, 2047, 4096)["time_chunks"] > 1
    assert sp.spiir_host_geometry(16, 128, 1, 2047, 128)["time_chunks"] == 1


def test_lane_mapping_many_templates(sp):
    # at least 16 x 148 templates: 32..64 filters take a quarter warp per template (four templates per warp), 65..128
    # half a warp (two templates per warp)
    g = sp.spiir_host_geometry(4096, 64, 1, 100, 1024)
    assert (g["F"], g["lanes_per_template"]) == (8, 8)
    g = sp.spiir_host_geometry(4096, 32, 1, 100, 1024)
    assert (g["F"], g["lanes_per_template"]) == (4, 8)
    g = sp.spiir_host_geometry(4096, 65, 1, 100, 1024)
    assert (g["F"], g["lanes_per_template"]) == (5, 16)
    g = sp.spiir_host_geometry(4096, 128, 1, 100, 1024)
    assert (g["F"], g["lanes_per_template"]) == (8, 16)
    g = sp.spiir_host_geometry(4096, 129, 1, 100, 1024)
    assert (g["F"], g["lanes_per_template"]) == (5, 32)
    g = sp.spiir_host_geometry(2367, 64, 1, 100, 1024)
    assert (g["F"], g["lanes_per_template"]) == (2, 32)


def test_layout_is_a_permutation_and_avoids_bank_conflicts(sp):
    from paper_1702_02256_b200 import inputs
    b = inputs.config(1, n_templates=16).banks[0]
    lay = sp.spiir_host_layout(b.a1, b.b0, b.delays, True)
    nat = sp.spiir_host_layout(b.a1, b.b0, b.delays, False)
    for L_ in (lay, nat):
        pos = L_["pos"]
        assert pos.shape == (16, 256) and len(np.unique(pos)) == pos.size          # injective
        assert pos.min() >= 0 and pos.max() < L_["G"] * L_["F"] * 32
        c = L_["coef"][pos.ravel()]
        np.testing.assert_array_equal(c[:, 0] + 1j * c[:, 1], b.a1.ravel())
        np.testing.assert_array_equal(c[:, 2] + 1j * c[:, 3], b.b0.ravel())
        np.testing.assert_array_equal(L_["dly"][pos.ravel()], b.delays.ravel())
        # template t lives in group t (one warp per template for L = 256)
        np.testing.assert_array_equal(pos // (L_["F"] * 32), np.arange(16)[:, None] * np.ones((1, 256), int))
    assert nat["conflict_degree"] > 2.0          # random delays: ~2.5 bank-group collisions per quarter warp
    assert lay["conflict_degree"] < 1.4          # permuted: only the class imbalance of 256 random delays is left
    assert lay["conflict_degree"] >= 1.0


def test_layout_small_templates_share_a_warp(sp):
    from paper_1702_02256_b200 import inputs
    b = inputs.config(2, n_templates=100, n_filters=8).banks[0]
    lay = sp.spiir_host_layout(b.a1, b.b0, b.delays, True)
    assert (lay["F"], lay["LPT"]) == (4, 2)
    assert lay["G"] == (100 + 15) // 16                    # 16 templates of 2 lanes per warp
    pos = lay["pos"]
    lane = pos % 32
    np.testing.assert_array_equal(lane // 2, (np.arange(100) % 16)[:, None] * np.ones((1, 8), int))
    # padding slots carry zero coefficients
    used = np.zeros(lay["dly"].size, bool)
    used[pos.ravel()] = True
    assert np.all(lay["coef"][~used] == 0)


def test_geometry_of_the_baseline_configs(sp):
    g1 = sp.spiir_host_geometry(1024, 256, 1, 4095, 4096)
    assert g1["time_chunks"] == 1 and g1["launches"] == 1
    assert g1["warps_per_cta"] == 7 and g1["grid"] == 147                       # one CTA per SM, 7 templates each
    assert g1["time_tile"] == 4096 and g1["smem_bytes"] <= 232448
    assert g1["smem_bytes"] == 16 * (4096 + 4096 + 32) + 16                      # four shifted window copies + mbarrier
    gm = sp.spiir_host_geometry(64, 1024, 1, 4095, 4096)                          # multi-warp templates: + reduction tiles
    assert gm["smem_bytes"] == 16 * (4096 + 4096 + 32) + 16 + gm["warps_per_cta"] * (32 * 9 + 64) * 16
    g0 = sp.spiir_host_geometry(16, 128, 1, 2047, 4096)
    assert g0["time_chunks"] > 8 and g0["launches"] == 3                        # 16 warps of work -> chunked scan
    g4 = sp.spiir_host_geometry(16384, 256, 2, 2047, 2048)
    assert g4["time_chunks"] == 1 and g4["warps_per_cta"] == 8
    assert g4["grid"] <= 2 * 148 + 2                                            # persistent CTAs loop over groups
    assert 2 * (g4["smem_bytes"] + 1024) <= 233472                              # two CTAs share an SM
    # forcing chunks / forbidding them
    assert sp.spiir_host_geometry(1024, 256, 1, 4095, 4096, time_chunks=4)["time_chunks"] == 4
    assert sp.spiir_host_geometry(16, 128, 1, 2047, 4096, time_chunks=1)["time_chunks"] == 1
    # a long block is tiled in time when the window would not fit shared memory
    g = sp.spiir_host_geometry(1024, 256, 1, 4095, 65536, time_chunks=1)
    assert g["time_tile"] < 65536 and g["time_tile"] % 16 == 0 and g["smem_bytes"] <= 232448
    with pytest.raises(sp.SpiirError):
        sp.spiir_host_geometry(4, 8, 1, 100000, 256)                            # delay beyond the window limit


def test_kaiser_taps_against_numpy(sp):
    """Same closed form as the paper's Eq. 9 design (readings R1-R3), evaluated with numpy.kaiser."""
    N, beta, fc = 192, 5.0, 0.25
    h = sp.spiir_kaiser_taps(N, beta, fc).astype(np.float64)
    n = np.arange(N) - (N - 1) / 2
    ref = np.kaiser(N, beta) * 2 * fc * np.sinc(2 * fc * n)
    ref /= ref.sum()
    np.testing.assert_allclose(h, ref, rtol=0, atol=1.6e-8)      # half an ulp of the largest tap (0.45)
    assert abs(h.sum() - 1.0) < 1e-6
    np.testing.assert_array_equal(h, h[::-1])
    for (N2, b2, c2) in ((32, 3.0, 0.2), (384, 10.0, 0.25), (2, 0.0, 0.5)):
        h2 = sp.spiir_kaiser_taps(N2, b2, c2).astype(np.float64)
        n2 = np.arange(N2) - (N2 - 1) / 2
        r2 = np.kaiser(N2, b2) * 2 * c2 * np.sinc(2 * c2 * n2)
        np.testing.assert_allclose(h2, r2 / r2.sum(), rtol=0, atol=1e-7)


def test_product_path_does_not_touch_the_oracle():
    """The package, bench.py's default arm and the C sources never import or link oracle/."""
    pkg = os.path.join(ROOT, "paper_1702_02256_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), f
                assert "spiir_oracle" not in text, f
