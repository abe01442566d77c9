"""Host logic: seeded input recipe and the update counter (the unit of BASELINE.json's metric)."""
import os

import numpy as np

from paper_1702_02256_b200 import inputs

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def read_table(name):
    rows = []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                rows.append(line.split())
    return rows


def test_update_counter_against_paper_table3():
    """PAPER.md:233-244 Table 3: 1024 filters split equally over H rates; the CPU filtering time
    relative to one rate must follow the 12*N*M*R model: (1/H) sum_h 2^-h."""
    rows = {int(r[0]): float(r[1]) for r in read_table("paper_table3_filtering_seconds.txt")}
    single = inputs.updates_per_block([1024], 4096, 1, 4096)
    assert single == 4096 * 1024 * 4096
    for H, secs in rows.items():
        ours = inputs.updates_per_block([1024 // H] * H, 4096, 1, 4096) / single
        assert abs(ours - secs / rows[1]) < 0.03 * ours, (H, ours, secs / rows[1])


def test_cost_model_statement():
    """half the filters at R/2 reduces the cost by 25 %."""
    vals = dict((r[0], float(r[1])) for r in read_table("paper_cost_model.txt"))
    full = inputs.updates_per_block([512], 7, 1, 64)
    half = inputs.updates_per_block([256, 256], 7, 1, 64)
    assert half / full == vals["half_filters_at_half_rate_cost_ratio"]


def test_config_shapes_and_distributions():
    w = inputs.config(0)
    b = w.banks[0]
    assert b.a1.shape == (16, 128) and b.a1.dtype == np.complex64 and b.delays.dtype == np.int32
    mag = np.abs(b.a1.astype(np.complex128))
    assert mag.min() >= 0.9 - 1e-6 and mag.max() <= 0.9999 + 1e-6
    assert b.delays.min() >= 0 and b.delays.max() <= 2047
    assert w.updates_per_block() == 16 * 128 * 4096
    x = w.strain(0)
    assert x.shape == (1, 4096) and x.dtype == np.float32
    assert np.array_equal(x, inputs.config(0).strain(0)) and not np.array_equal(x, w.strain(1))
    assert abs(np.std(np.abs(b.b0)) - 1e-3 * np.sqrt(1 - np.pi / 4)) < 1e-4   # Rayleigh spread of 1e-3*CN(0,1)


def test_config_update_counts_match_survey():
    assert inputs.config(1, n_templates=4).updates_per_block() == 4 * 256 * 4096
    w3 = inputs.config(3, n_templates=2)
    assert [b.a1.shape[1] for b in w3.banks] == [8, 16, 32, 48, 64, 48, 40]
    assert w3.updates_per_block() == 2 * 147968
    assert all(b.delays.max() <= b.rate_hz - 1 for b in w3.banks)
    w4 = inputs.config(4, n_templates=8)
    assert w4.n_streams == 2 and w4.strain(0).shape == (2, 2048)
    assert not np.array_equal(w4.strain(0)[0], w4.strain(0)[1])
    w2 = inputs.config(2, n_templates=16, n_filters=4)
    assert w2.banks[0].a1.shape == (16, 4) and np.abs(w2.banks[0].a1).max() <= 0.999 + 1e-6


def test_shard_templates_covers_everything_once():
    for T in (1, 7, 1024, 16384):
        for W in (1, 2, 3, 8):
            spans = [inputs.shard_templates(T, W, r) for r in range(W)]
            assert spans[0][0] == 0 and spans[-1][1] == T
            assert all(spans[i][1] == spans[i + 1][0] for i in range(W - 1))
            sizes = [hi - lo for lo, hi in spans]
            assert max(sizes) - min(sizes) <= 1
