"""The seeded input generators: known answers and the recipe's stated properties."""
import os

import numpy as np

from workloads import splitmix64_u64, uniform01, make_config, make_xs, single_sweep_case, paper_shaped

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_splitmix64_known_answer():
    # reference outputs of splitmix64 seeded with 0 (Vigna's public-domain generator)
    got = [int(splitmix64_u64(0, i)) for i in range(3)]
    assert got[0] == 0xE220A8397B1DCDAF
    assert got[1] == 0x6E789E6AA1B965F4
    assert got[2] == 0x06C45D188009454F
    u = uniform01(123, np.arange(1000))
    assert 0.0 <= u.min() and u.max() < 1.0 and abs(u.mean() - 0.5) < 0.05


def test_water_mean_free_path_matches_paper():
    # 13.9 mm at 20 keV and 60.6 mm at 100 keV fix a = 4468, b = 0.1605 for water
    for line in open(os.path.join(GOLD, "paper_facts.txt")):
        if line.startswith("mfp_mm"):
            _, e, mfp = line.split()
            sig = 4468.0 * float(e) ** -3 + 0.1605
            assert abs(10.0 / sig - float(mfp)) < 0.05


def test_xs_recipe():
    E, st, ss = make_xs(1910113351, 19, 3, 10.0, 100.0)
    assert E[0] > E[-1] and abs(E[0] - (100 - 90 / 38)) < 1e-12
    assert (np.diff(st, axis=1) > 0).all()                        # sigma_t rises as energy falls
    for gp in range(19):
        assert (ss[:, :, gp, :gp] == 0).all()                      # downscatter only
        c = 0.3 + 0.6 * (E[gp] - E[-1]) / (E[0] - E[-1])
        assert np.allclose(ss[:, 0, gp, :].sum(-1), c * st[:, gp])   # total out-scatter = c sigma_t
    assert np.allclose(ss[:, 1], 0.3 * ss[:, 0]) and np.allclose(ss[:, 3], 0.027 * ss[:, 0])


def test_config_shapes():
    w0 = make_config(0)
    assert (w0.nx, w0.G, w0.L, w0.sn, w0.fixed_iters) == (8, 1, 0, 2, 10)
    assert w0.sources[0].volume.sum() == 8.0
    w1 = make_config(1)
    assert (w1.nx, w1.G, w1.L, w1.sn) == (32, 19, 3, 8) and set(np.unique(w1.material)) == {0, 2}
    w2 = make_config(2)
    assert set(np.unique(w2.material)) == {0, 1, 2, 3} and w2.density.max() == np.float32(1.85)
    s = single_sweep_case(2, groups=(0, 5), fixed_iters=2)
    assert s.G == 2 and s.sigma_s.shape == (4, 4, 2, 2) and s.sigma_s[2, 0, 0, 1] == w2.sigma_s[2, 0, 0, 5]
    p = paper_shaped()
    assert (p.nx, p.ny, p.nz, p.G, p.L, p.sn) == (64, 64, 16, 90, 0, 6)


def test_config3_density_noise():
    w = make_config(3)
    base = np.array([0.0012, 0.3, 1.0, 1.85])[w.material]
    r = w.density.astype(float) / base
    assert r.min() >= 0.95 - 1e-6 and r.max() <= 1.05 + 1e-6 and abs(r.mean() - 1) < 1e-3
