"""The seeded generator: determinism, row addressability, truth table."""
import numpy as np

import gen


def test_rows_are_addressable_and_deterministic():
    cfg = gen.get_config(1)
    a = gen.make_array(cfg, threads=1)
    b = gen.make_array(cfg, threads=4)
    assert a.dtype == np.float32 and a.shape == (64, 16384)
    assert np.array_equal(a, b)
    rows = [0, 17, 63]
    assert np.array_equal(gen.make_rows(cfg, rows), a[rows])
    assert np.array_equal(gen.make_array(cfg, row_lo=10, row_hi=20), a[10:20])


def test_truth_table_is_injected():
    cfg = gen.get_config(1)
    clean = gen.custom_config(cfg.n_dm, cfg.n_t, cid=cfg.cid)      # same seeds, no pulses
    a, n = gen.make_array(cfg), gen.make_array(clean)
    diff = a.astype(np.float64) - n
    tab = gen.pulse_table(cfg)
    assert [p.width for p in tab] == [1, 2, 4, 8, 16]
    mask = np.zeros(a.shape, bool)
    for p in tab:
        assert np.allclose(diff[p.row, p.start:p.start + p.width], p.amp, atol=1e-5)
        mask[p.row, p.start:p.start + p.width] = True
    assert np.all(diff[~mask] == 0)
    assert sorted({p.row for p in tab}) == gen.pulse_rows(cfg)


def test_config_shapes_match_baseline():
    shapes = {1: (64, 16384), 2: (1024, 131072), 3: (6000, 262144), 4: (2048, 262144), 5: (4096, 524288)}
    for cid, (n_dm, n_t) in shapes.items():
        c = gen.get_config(cid)
        assert (c.n_dm, c.n_t) == (n_dm, n_t)
        assert len(gen.pulse_table(c)) == {1: 5, 2: 50, 3: 200, 4: 500, 5: 1000}[cid]
    assert gen.get_config(5).n == 2 ** 31
    assert gen.get_config(4).sigma_mode == "linear" and gen.get_config(5).nmax == (8, 32, 128, 512)


def test_c2_offset_noise_and_c3_smear():
    c2 = gen.get_config(2)
    r = gen.make_rows(c2, [5]).astype(np.float64)
    assert abs(r.mean() - 100) < 0.5 and abs(r.std() - 20) < 0.5
    c3 = gen.get_config(3)
    p = gen.pulse_table(c3)[0]
    rows = [q for q in range(p.row - 3, p.row + 4) if 0 <= q < c3.n_dm]
    assert set(rows) <= set(gen.pulse_rows(c3))
