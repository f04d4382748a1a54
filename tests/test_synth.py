"""The seeded input generator (paper_2509_25110_b200/synth.py): grids, noise, slices (R7-R11, R22)."""
import numpy as np

from paper_2509_25110_b200 import synth


def test_splitmix64_reference_outputs():
    # the public-domain splitmix64 step: first output for state 1234
    assert synth._mix_int(1234) == 0xBB0CF61B2F181CDB
    assert synth.stream_base(1234, 0) == 0xBB0CF61B2F181CDB
    u = synth.uniform_pm1(1234, 0, 0, 4)
    assert np.allclose(u, [0.23510400924273411, 0.39626839495455268, -0.21405092369648715,
                           -0.14091297765222555], rtol=0, atol=1e-16)
    big = synth.uniform_pm1(1234, 5, 0, 200000)
    assert big.min() >= -1.0 and big.max() < 1.0
    assert abs(big.mean()) < 5e-3 and abs(big.var() - 1 / 3) < 5e-3
    assert np.array_equal(synth.uniform_pm1(1234, 5, 1000, 50), big[1000:1050])   # counter-based


def test_grids_match_the_config_statements():
    for cfg in synth.CONFIGS:
        k, tau = cfg.k(), cfg.tau()
        assert k.size == cfg.n_k and tau.size == cfg.n_tau
        assert k[0] == cfg.k_lo and k[-1] == cfg.k_hi
        assert np.all(np.diff(k) > 0) and np.all(np.diff(tau) > 0)
        assert np.allclose(np.diff(np.log(k)), np.log(cfg.k_hi / cfg.k_lo) / (cfg.n_k - 1), rtol=1e-9)
        assert tau[0] == 200.0 and tau[cfg.n_tau_uniform - 1] == 400.0 and tau[-1] == cfg.tau0 - 1.0
        assert np.allclose(np.diff(tau[:cfg.n_tau_uniform]), 200.0 / (cfg.n_tau_uniform - 1))
        assert np.all(tau < cfg.tau0)
        assert cfg.l_list()[0] == 2 and cfg.l_list()[-1] == cfg.l_max
    c1 = synth.CONFIGS[1]
    assert (c1.n_l, c1.n_k, c1.n_tau) == (2499, 3000, 1200)
    assert synth.CONFIGS[3].n_batch == 64 and synth.CONFIGS[4].n_src == 3


def test_sources_slices_and_noise_level():
    cfg = synth.CONFIGS[0]
    S_T, S_E, S_P = synth.sources(cfg)
    assert S_P is None and S_T.shape == (cfg.n_k, cfg.n_tau) and S_T.flags.c_contiguous
    a, b, _ = synth.sources(cfg, k_slice=slice(37, 90, 5))
    assert np.array_equal(a, S_T[37:90:5]) and np.array_equal(b, S_E[37:90:5])
    c_T, c_E, _ = synth.sources(cfg, noise=False)
    r = S_T / c_T - 1
    assert np.max(np.abs(r)) <= 1e-3 * (1 + 1e-12) and np.std(r) > 4e-4
    cfg2 = synth.Config(9, "t", 2, 50, 40, 1e-4, 0.3, 20, 10, True)
    _, _, P = synth.sources(cfg2)
    assert P is not None and P.shape == (40, 30) and np.all(P > 0)


def test_emulator_batch_parameter_ranges():
    cfg = synth.CONFIGS[3]
    seen = set()
    for c in range(64):
        p = synth.cosmology(cfg, c)
        assert 15 <= p.sigma < 25 and 260 <= p.mu < 300 and 0.55 <= p.c_s < 0.6
        assert 1.9e-9 <= p.A_s < 2.3e-9 and 0.94 <= p.n_s < 0.99
        seen.add(round(p.sigma, 9))
    assert len(seen) == 64
    assert synth.cosmology(synth.CONFIGS[1], 0) == synth.Cosmology()
    P = synth.primordial_power(synth.CONFIGS[1])
    k = synth.CONFIGS[1].k()
    assert np.allclose(P, 2.1e-9 * (k / 0.05) ** -0.035, rtol=1e-14)
