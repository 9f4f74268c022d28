"""Host-side checks of the seeded synthetic workloads (paper_1909_07321_b200/inputs.py)."""
import numpy as np
import pytest

from paper_1909_07321_b200 import inputs


@pytest.mark.parametrize("cfg,P,C,N", [(1, 1, 8, 1000), (2, 1, 64, 4096), (5, 1, 512, 256)])
def test_single_wave_configs(cfg, P, C, N):
    wl = inputs.make_config(cfg)
    assert len(wl.waves) == P
    w = wl.waves[0]
    assert (w.n_chan, w.n_poles, w.n_E) == (C, 20 * C, N)
    assert w.W.dtype == np.float64 and w.W.flags.c_contiguous
    assert np.all(np.diff(w.E_k) >= 0)
    assert np.all(inputs.min_pole_distance(w.energies, w.E_k) >= inputs.CLEARANCE_RYD)
    assert wl.sha256() == inputs.make_config(cfg).sha256()          # seeded: same bits every time
    assert wl.counted_flop() == float(N) * C * C * 20 * C


def test_config3_shared_mesh_clear_of_all_waves():
    wl = inputs.make_config(3, n_E=256)
    assert len(wl.waves) == 8
    for w in wl.waves:
        assert w.energies is wl.waves[0].energies
        assert (w.n_chan, w.n_poles) == (256, 5120)
        assert np.all(inputs.min_pole_distance(w.energies, w.E_k) >= inputs.CLEARANCE_RYD)
    assert not np.array_equal(wl.waves[0].W, wl.waves[1].W)


def test_config4_ragged():
    shapes = inputs.config_shapes(4)
    assert len(shapes) == 32
    chans = [s[0] for s in shapes]
    assert min(chans) >= 16 and max(chans) <= 400 and len(set(chans)) > 16
    assert all(s[1] == 20 * s[0] and s[2] == 512 for s in shapes)
    wl = inputs.make_config(4, n_E=16)
    assert [w.n_chan for w in wl.waves] == chans
    for w in wl.waves:
        assert np.all(inputs.min_pole_distance(w.energies, w.E_k) >= inputs.CLEARANCE_RYD)
        assert w.energies[0] == pytest.approx(0.01, abs=5e-3) and w.energies[-1] == pytest.approx(50.0, abs=5e-3)


def test_nudge_rule():
    poles = np.array([1.0, 1.0015, 5.0])
    e = np.array([0.5, 0.9995, 1.0005, 1.0012, 4.9999, 5.0, 7.0])
    out = inputs.nudge_off_poles(e, poles)
    assert out[0] == 0.5 and out[-1] == 7.0                         # clear points untouched
    assert np.all(inputs.min_pole_distance(out, np.sort(poles)) >= 1e-3)
    assert out[1] <= 0.999 and out[2] <= 0.999 and out[3] >= 1.0025 - 1e-12   # merged interval [0.999, 1.0025]: nearer end
    assert out[4] < 4.9991 and out[5] >= 5.001                      # tie goes up
    assert np.all(np.abs(out - e) <= 2.6e-3)


def test_meshes():
    m = inputs.linear_mesh(0.1, 10.0, 1000)
    assert m[0] == 0.1 and abs(m[-1] - 10.0) < 1e-12 and np.allclose(np.diff(m), 9.9 / 999)
    g = inputs.geometric_mesh(0.01, 50.0, 512)
    assert g[0] == 0.01 and abs(g[-1] - 50.0) < 1e-9 and np.allclose(g[1:] / g[:-1], (5000.0) ** (1 / 511))


def test_sample_energy_indices():
    w = inputs.make_wave(3, 4, 80, 100)
    idx = inputs.sample_energy_indices(w)
    assert idx[0] == 0 and idx[-1] == 99 and len(idx) == len(set(idx)) and len(idx) <= 8
    assert int(np.argmin(inputs.min_pole_distance(w.energies, w.E_k))) in idx
