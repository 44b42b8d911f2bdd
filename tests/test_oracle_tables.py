"""Pins for the oracle's integer tables and loop bounds (O1, O2, n_images) and for the
input shapes -- against the paper's printed values, closed forms and exact rational
arithmetic, never against the oracle itself.  CPU only."""
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle as O
import workloads as W


def _read_kv(path):
    out = {}
    for line in open(path):
        line = line.split("#")[0].strip()
        if line:
            k, *v = line.split()
            out[k] = v
    return out


# ------------------------------------------------------------------ paper constants
def test_dispersion_constant_matches_paper(golden_dir):
    kv = _read_kv(os.path.join(golden_dir, "paper_constants.txt"))
    # PAPER.md:45 prints 4.15 ms; reading A1 uses 4.148808e-3 s, which rounds to it
    assert round(O.K_DM * 1e3, 2) == float(kv["dispersion_ms"][0])
    assert O.K_DM == 4.148808e-3


def test_sweep_worked_example(golden_dir):
    """DM 2000, 256 MHz at 1.4 GHz -> 'roughly 2 seconds' (P3: same order)."""
    kv = _read_kv(os.path.join(golden_dir, "paper_constants.txt"))
    fc, bw = float(kv["sweep_fc_ghz"][0]), float(kv["sweep_bw_mhz"][0]) / 1e3
    f = np.array([fc - bw / 2, fc + bw / 2]) * 1e9
    d = O.delay_table(f, [float(kv["sweep_dm"][0])], 1e-3)[0]      # 1 ms integrations
    sweep_s = d[0] * 1e-3
    assert d[1] == 0
    assert 0.5 * float(kv["sweep_s"][0]) < sweep_s < 1.5 * float(kv["sweep_s"][0])
    assert abs(sweep_s - 1.575) < 2e-3                               # closed form by hand


def test_table1_data_rates_fix_shape_and_dtype(golden_dir):
    """P4: Table 1 rates = 351 bl x nchan x 2 pol x 8 B / t_int  => complex64 [.,351,nchan,2]."""
    for line in open(os.path.join(golden_dir, "paper_table1_rates.txt")):
        if line.startswith("#"):
            continue
        _, nchan, t_ms, rate = line.split()
        got = 351 * int(nchan) * 2 * 8 / (float(t_ms) * 1e-3) / 1e6
        assert abs(got - float(rate)) / float(rate) < 0.05
    cfg = W.get_config("lband")
    assert (cfg.nbl, cfg.nchan, cfg.npol) == (351, 256, 2)
    row = W.noise_rows(cfg, [0])
    assert row.dtype == np.complex64 and row.shape == (1, 351, 256, 2)


# ------------------------------------------------------------------ O1 delay table
def test_delay_closed_form_properties():
    """P1: DM 0 -> 0; top channel 0; non-increasing in f; any channel order."""
    for name in ("tiny", "lband", "sband", "hires"):
        cfg = W.get_config(name)
        f = W.channel_freqs_hz(cfg)
        d = O.delay_table(f, W.dm_list(cfg), cfg.inttime_s)
        assert d.dtype == np.int32 and d.shape == (cfg.ndm, cfg.nchan)
        assert (d[0] == 0).all()
        assert (d[:, np.argmax(f)] == 0).all()
        assert (d >= 0).all()
        assert (np.diff(d, axis=1) <= 0).all()          # f ascending -> delay non-increasing
        assert (np.diff(d, axis=0) >= 0).all()          # DM ascending -> delay non-decreasing
        perm = np.random.default_rng(0).permutation(cfg.nchan)
        assert (O.delay_table(f[perm], W.dm_list(cfg), cfg.inttime_s) == d[:, perm]).all()


def test_delay_golden_tiny(golden_dir):
    """P2: survey-derived rows for config 1 (independent script, readings A1-A4)."""
    kv = _read_kv(os.path.join(golden_dir, "tiny_delays.txt"))
    cfg = W.get_config("tiny")
    f = W.channel_freqs_hz(cfg)
    assert f[0] == 1.0078125e9 and f[-1] == 1.4921875e9
    assert O.delay_table(f, [50.0], cfg.inttime_s)[0].tolist() == [int(v) for v in kv["dm50"]]
    d = O.delay_table(f, W.dm_list(cfg), cfg.inttime_s)
    assert d.max(axis=1).tolist() == [int(v) for v in kv["maxdelay_per_trial"]]


def test_max_delay_and_image_counts_golden(golden_dir):
    for line in open(os.path.join(golden_dir, "config_max_delays.txt")):
        if line.startswith("#"):
            continue
        name, maxd, nimg = line.split()
        cfg = W.get_config(name)
        d = O.delay_table(W.channel_freqs_hz(cfg), W.dm_list(cfg), cfg.inttime_s)
        assert int(d.max()) == int(maxd)
        total = sum(O.n_images(cfg.nint, int(d[i].max()), dt)
                    for i in range(cfg.ndm) for dt in cfg.dt_list)
        assert total == int(nimg)


@pytest.mark.parametrize("name", ["tiny", "lband", "hires"])
def test_delay_exact_rational(name):
    """The float64 table equals round-half-up of the EXACT rational value of the same
    expression (Fractions of the float inputs), and no entry is within 1e-7 of a tie."""
    cfg = W.get_config(name)
    f = W.channel_freqs_hz(cfg)
    dms = W.dm_list(cfg)
    d = O.delay_table(f, dms, cfg.inttime_s)
    fg = [Fraction(float(v)) / Fraction(10) ** 9 for v in f]
    fmax = max(fg)
    K, tint = Fraction(O.K_DM), Fraction(cfg.inttime_s)
    step = max(1, cfg.ndm // 8)
    for i in list(range(0, cfg.ndm, step)) + [cfg.ndm - 1]:
        for c in range(0, cfg.nchan, max(1, cfg.nchan // 64)):
            x = K * Fraction(float(dms[i])) * (1 / (fg[c] * fg[c]) - 1 / (fmax * fmax)) / tint
            exact = (x + Fraction(1, 2)).__floor__()
            frac = x - x.__floor__()
            assert abs(frac - Fraction(1, 2)) > Fraction(1, 10 ** 7)
            assert d[i, c] == exact


def test_n_images_bounds():
    # (j+1)*dt <= nint - maxdelay  (A16); trailing partial bin dropped (A6)
    assert O.n_images(64, 0, 1) == 64
    assert O.n_images(64, 31, 1) == 33
    assert O.n_images(64, 31, 2) == 16
    assert O.n_images(64, 64, 1) == 0 and O.n_images(64, 70, 1) == 0
    assert O.n_images(1024, 624, 8) == 50
    assert O.n_images(1024, 624, 8, span=400) == 50 and O.n_images(1024, 0, 8, span=400) == 50
    assert O.n_images(1024, 0, 1, span=400) == 400


# ------------------------------------------------------------------ O2 cell table
def test_cell_table_exact_rational_and_range():
    """Cells equal round-half-up of the exact rational u_lambda/du; all inside the
    central 2/3 of the grid for cell = 1/(3 max|uv|) (A13)."""
    for name in ("tiny", "lband"):
        cfg = W.get_config(name)
        f = W.channel_freqs_hz(cfg)
        uvw = W.baseline_uvw_m(cfg)
        cell = W.default_cell_rad(cfg, uvw)
        iu, iv, keep = O.cell_table(uvw, f, cfg.npix, cell)
        assert keep.all()
        assert np.abs(iu).max() <= cfg.npix // 3 + 1 and np.abs(iv).max() <= cfg.npix // 3 + 1
        rng = np.random.default_rng(1)
        du = Fraction(1.0 / (cfg.npix * cell))          # du is ONE float64 in the definition
        for _ in range(200):
            b, c = int(rng.integers(cfg.nbl)), int(rng.integers(cfg.nchan))
            for col, tab in ((0, iu), (1, iv)):
                ul = Fraction(float(uvw[b, col] * f[c] / O.C_LIGHT))
                x = ul / du
                # the float64 quotient is within 1 ulp of x: exact unless x is within 1e-9 of a tie
                frac = x - x.__floor__()
                if abs(frac - Fraction(1, 2)) > Fraction(1, 10 ** 9):
                    assert tab[b, c] == (x + Fraction(1, 2)).__floor__()


def test_cell_table_drops_offgrid_and_flagged():
    uvw = np.array([[10.0, 5.0, 0.0], [400.0, -20.0, 1.0], [-30.0, 390.0, 2.0], [-320.0, 0.0, 0.0]])
    f = np.array([1.0e9, 1.2e9])
    npix = 64
    # du chosen so that u = 400 m at 1.2 GHz lands beyond +N/2 and -320 m at 1.0 GHz exactly at -N/2
    du = 320.0 * 1.0e9 / O.C_LIGHT / 32.0
    cell = 1.0 / (npix * du)
    iu, iv, keep = O.cell_table(uvw, f, npix, cell)
    assert iu[3, 0] == -32 and keep[3, 0]              # -N/2 is inside [-N/2, N/2)
    assert iu[1, 0] == 40 and not keep[1, 0]           # off grid: dropped, never wrapped
    assert not keep[2, 0] and keep[0].all()
    w = np.array([1.0, 0.0], dtype=np.float32)
    _, _, keep_w = O.cell_table(uvw, f, npix, cell, w)
    assert not keep_w[:, 1].any() and (keep_w[:, 0] == keep[:, 0]).all()
