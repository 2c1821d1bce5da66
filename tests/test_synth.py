"""Host logic of the seeded workload generators."""
import numpy as np

from paper_2510_19047_b200 import synth


def test_shapes_and_determinism():
    w = synth.scaled(synth.WORKLOADS["cfg3"], Nt=256, Nf=128)
    c1, w1, g1 = synth.make_data(w)
    c2, w2, g2 = synth.make_data(w)
    assert c1.shape == (2, 256, 128, 2) and w1.shape == (2, 256, 128) and g1.shape == (256,)
    assert c1.dtype == np.float32 and g1.dtype == np.uint8
    assert np.array_equal(c1, c2) and np.array_equal(w1, w2) and np.array_equal(g1, g2)
    p = synth.make_templates(w, 1000)
    assert p.shape == (1000, 8) and p.dtype == np.float64
    assert np.all((p[:, 0] >= 5) & (p[:, 0] <= 100)) and np.all(p[:, 1] >= 0)
    assert np.allclose(np.linalg.norm(p[:, 3:7], axis=1), 1.0)


def test_noise_matches_weights():
    # E|D|^2 = 2/W per pixel
    w = synth.scaled(synth.WORKLOADS["cfg2"], Nt=512, Nf=256)
    c, wt, g = synth.make_data(w)
    p2 = c[..., 0].astype(np.float64) ** 2 + c[..., 1].astype(np.float64) ** 2
    ok = wt > 0
    r = np.mean(p2[ok] * wt[ok])
    assert abs(r / 2 - 1) < 0.01
    assert np.all(wt[:, :, 0] == 0) and np.all(c[:, :, 0] == 0)       # k = 0 carries no weight
    assert np.all(g == 1)


def test_gap_duty_cycle():
    w = synth.WORKLOADS["cfg3"]
    g = synth.gap_mask(w, np.random.default_rng(w.seed))
    assert 0.80 < g.mean() < 0.95
    assert synth.gap_mask(synth.WORKLOADS["cfg1"], np.random.default_rng(0)).all()


def test_cfg4_has_merging_templates():
    w = synth.WORKLOADS["cfg4"]
    p = synth.make_templates(w, 5000)
    Tobs = w.Nt * w.DT
    assert np.all(p[::5, 1][:1000] <= Tobs) and np.all(p[::5, 0][:1000] >= 30)
    assert len(synth.injection_params(synth.WORKLOADS["cfg5"])) == 5
