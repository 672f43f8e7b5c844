"""Seeded input generators: determinism, shapes, value structure."""
import numpy as np

from paper_2112_11991_b200 import workloads as wl


def test_c1_is_seeded_and_shaped(c1):
    again = wl.config1()
    assert np.array_equal(c1.series, again.series) and np.array_equal(c1.templates, again.templates)
    assert c1.series.dtype == np.float32 and c1.series.size == 1 << 17
    assert c1.templates.shape == (64, 5) and c1.templates.dtype == np.float64
    assert c1.templates[0].tolist() == [60.0, 0.5, 1.0, 0.0, 0.0]
    t = c1.templates[1:]
    assert t[:, 0].min() >= 40 and t[:, 0].max() <= 90 and t[:, 1].min() >= 0 and t[:, 1].max() <= 1
    assert abs(float(c1.series.std()) - 1.0) < 0.02


def test_small_variants_of_c2_c3_c4_c5():
    c2 = wl.config2(n_templates=16, log2n=16)
    assert c2.templates.shape == (16, 5) and c2.true_ids == (0, 1, 2) and np.all(c2.templates[:, 3:] == 0)
    c3 = wl.config3(n_templates=8, log2n=16)
    q = c3.series * 32.0
    assert np.array_equal(q, np.rint(q)) and q.min() >= -128 and q.max() <= 127   # 8-bit codes
    c4 = wl.config4(n_templates=8, log2n=16, tau_scale=1 / 512)
    assert c4.templates[0, 3] == 0.08 and c4.templates[0, 4] == 1.2
    assert c4.templates[1:, 3].max() <= 0.1 and c4.templates[1:, 3].min() >= 0
    c5 = wl.config5(log2n=16, n_circ=4, n_ell=4)
    assert np.all(c5.templates[:4, 3:] == 0) and np.all(c5.templates[4:, 3] > 0)
    beta = c5.templates[:, 1] * 2 * np.pi / c5.templates[:, 0]
    assert beta.min() >= 0.001 and beta.max() <= 0.1


def test_paper_shaped_workloads_small():
    """the paper's own simulation shape (Table 2) and a Terzan-5-length series, scaled down."""
    p = wl.config_paper(log2n=16, n_templates=8)
    assert p.tsamp == 256e-6 and p.templates.shape == (8, 5) and p.true_ids == (0,)
    assert p.templates[0, 0] == 8 * 3600.0 and p.templates[0, 3] == 0.1
    t = p.templates[1:]
    assert t[:, 0].min() >= 6 * 3600 and t[:, 0].max() <= 12 * 3600 and t[:, 1].max() <= 7 and t[:, 3].max() <= 0.1
    z = wl.config_terzan(log2n=16, n_templates=4)
    assert z.tsamp == 81.92e-6 and z.series.dtype == np.float32 and np.all(z.templates[:, 3:] == 0)
    assert 5 * z.t_obs <= z.templates[1:, 0].min() and z.templates[1:, 0].max() <= 10 * z.t_obs
    assert np.array_equal(z.series, wl.config_terzan(log2n=16, n_templates=4).series)
    # chunked injection = one-shot injection
    ref = wl.pulse_train(z.n_samples, z.tsamp, *z.pulsars[0][:7])
    noise = wl._rng(7).standard_normal(z.n_samples, dtype=np.float32)
    assert np.allclose(z.series - noise, ref.astype(np.float32), atol=1e-6)


def test_injection_is_inverse_of_the_gather_map():
    """s = t' - (Delta(t') - Delta(0)) solved for t': residual check (reading G3)."""
    s = np.linspace(0, 100, 1001)
    args = (37.0, 2.0, 0.4, 0.3, 1.0)
    t = wl.emission_times(s, *args)
    d, _ = wl._delay_and_rate(t, *args)
    d0, _ = wl._delay_and_rate(np.zeros(1), *args)
    assert np.max(np.abs(t - (d - d0[0]) - s)) < 1e-10


def test_shard_templates_covers_everything_once():
    for k in (1, 7, 64, 4097):
        for world in (1, 2, 3, 8):
            seen = []
            for r in range(world):
                first, count = wl.shard_templates(k, r, world)
                seen.extend(range(first, first + count))
            assert seen == list(range(k))
