"""The seeded generator: determinism, random access, structure."""
import numpy as np

from paper_2106_04649_b200 import configs, gen


def test_counter_rng_is_a_pure_function():
    a = gen.uniforms(7, 3, np.arange(10))
    b = gen.uniforms(7, 3, np.arange(10)[::-1])[::-1]
    np.testing.assert_array_equal(a, b)
    assert np.all((a >= 0) & (a < 1)) and len(np.unique(a)) == 10
    u = gen.uniforms(1, 1, np.arange(200000))
    assert abs(u.mean() - 0.5) < 5e-3 and abs(u.var() - 1 / 12) < 2e-3


def test_config_table_matches_baseline_json():
    shapes = [(101, 512, 0.004, 10.0, 1), (601, 2048, 0.004, 10.0, 1), (601, 2048, 0.004, 10.0, 601),
              (2001, 2048, 0.004, 10.0, 64), (3901, 4096, 0.002, 5.0, 256)]
    for k, (n, nt, dt, dx, nfoc) in enumerate(shapes):
        c = configs.get(k)
        assert (c.n, c.nt, c.dt, c.dx, c.nfoc, c.niter, c.eps, c.fmin, c.fmax) == (n, nt, dt, dx, nfoc, 16, 8, 5.0, 60.0)
        assert len(gen.focal_points(c)[0]) == nfoc
    assert configs.get(2).rseed == configs.get(1).seed            # "Same 601x601x2048 R as config 1"
    assert configs.get(3).noise_snr_db == 40.0


def test_R_is_causal_confined_and_blockwise_reproducible():
    cfg = configs.scaled(3, n=24, nt=256, nfoc=4, focal="fan:300")
    base = gen.base_traces(cfg)
    full = gen.R_full(cfg, base)
    assert full.dtype == np.float32 and full.shape == (24, 24, 256)
    assert np.all(full[:, :, 128:] == 0.0)                        # confined to [0, nt/2)
    blk = gen.R_block(cfg, base, [5, 17], [3, 4, 20])
    np.testing.assert_array_equal(blk, full[np.ix_([5, 17], [3, 4, 20])])
    assert np.abs(full - full.transpose(1, 0, 2)).max() > 0       # the noise makes R non-symmetric (G10 matters)
    noise = full - base[np.abs(np.arange(24)[:, None] - np.arange(24)[None, :])]
    snr = 20 * np.log10(np.sqrt((base[0, :128] ** 2).mean()) / noise[3, 3, :128].std())
    assert 35 < snr < 45


def test_first_arrivals():
    cfg = configs.get(0)
    gd, td = gen.first_arrivals(cfg)
    assert gd.shape == (1, 101, 512) and td.shape == (1, 101) and gd.dtype == np.float32 and td.dtype == np.float32
    r = np.argmin(td[0])
    assert r == 50 and abs(np.argmax(gd[0, r]) * cfg.dt - td[0, r]) <= cfg.dt
    frac = td.astype(np.float64) / cfg.dt + 0.5
    assert np.all(np.abs(frac - np.round(frac)) > 1e-4)           # no half-sample ties (G2c)


def test_device_twin_matches_numpy_generator():
    """gen.DeviceR (configs 3 / 4 are generated chunk by chunk on the device) == gen.R_block on a CPU torch device:
    bit-exact without noise; with noise the normals go through torch's log / cos / sin instead of numpy's, so allow
    one fp32 ulp of the trace peak."""
    import torch
    from paper_2106_04649_b200 import configs, gen
    for k, exact in ((4, True), (3, False)):
        cfg = configs.scaled(k, n=23, nt=128, nfoc=1, focal="single:300")
        base = gen.base_traces(cfg)
        shots, recs = np.array([0, 5, 22, 7]), np.array([3, 22, 0, 11, 12])
        ref = gen.R_block(cfg, base, shots, recs)
        got = gen.DeviceR(cfg, torch.device("cpu"), base).take(shots, recs).numpy()
        assert got.shape == ref.shape and got.dtype == np.float32
        if exact:
            np.testing.assert_array_equal(got, ref)
        else:
            assert np.abs(ref).max() > 0 and not np.array_equal(ref, gen.R_block(replace_noise(cfg), base, shots, recs))
            np.testing.assert_allclose(got, ref, rtol=0, atol=2e-7 * np.abs(ref).max())
        full = gen.DeviceR(cfg, torch.device("cpu"), base).take(np.arange(cfg.n)).numpy()
        np.testing.assert_allclose(full, gen.R_full(cfg, base), rtol=0, atol=0 if exact else 2e-7 * np.abs(ref).max())


def replace_noise(cfg):
    from dataclasses import replace
    return replace(cfg, noise_snr_db=None)


def test_first_arrivals_device_twin():
    import torch
    from paper_2106_04649_b200 import configs, gen
    cfg = configs.scaled(3, n=41, nt=256, nfoc=5, focal="fan:250")
    gd, td = gen.first_arrivals(cfg)
    gdt, tdt = gen.first_arrivals_torch(cfg, torch.device("cpu"), chunk=2)
    np.testing.assert_array_equal(tdt.numpy(), td)
    np.testing.assert_allclose(gdt.numpy(), gd, rtol=0, atol=2e-7)
    gdt2, tdt2 = gen.first_arrivals_torch(cfg, torch.device("cpu"), focs=[1, 4])
    np.testing.assert_array_equal(gdt2.numpy(), gdt.numpy()[[1, 4]])
