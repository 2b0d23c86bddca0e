"""The seeded workload generators: shapes, densities, seeds, structure."""
import numpy as np

from paper_1412_3387_b200 import inputs


def test_config1_exact():
    w = inputs.config(1)
    assert w.N == 4000 and abs(w.box[0] - 16.795962) < 1e-6 and w.rc == 2.5 and w.r_buff == 0.4
    assert abs(np.sum(w.vel ** 2) - (3 * w.N - 3) * 1.0) < 1e-8          # T = 1 exactly
    assert np.abs(w.vel.sum(axis=0)).max() < 1e-10                       # zero net momentum
    assert np.all(w.pos >= -0.5 * w.box) and np.all(w.pos < 0.5 * w.box)
    w2 = inputs.config(1)
    assert np.array_equal(w.pos, w2.pos) and np.array_equal(w.vel, w2.vel)   # seeded


def test_config2_recipe_small_replica():
    w = inputs.config(2, scale=(8 / 64) ** 3)                            # FCC 8^3 + jitter
    assert w.N == 4 * 8 ** 3 and w.precision == "mixed" and w.rc == 3.0
    assert abs(w.N / np.prod(w.box) - 0.8442) < 1e-12
    assert abs(np.sum(w.vel ** 2) / (3 * w.N - 3) - 1.2) < 1e-12
    ideal = inputs.fcc_positions(8, w.box[0])
    d = w.pos - ideal
    d -= w.box * np.rint(d / w.box)
    assert np.abs(d).max() <= 0.05 and np.abs(d).max() > 0.04            # jitter +-0.05 per axis


def test_full_size_counts():
    assert 4 * 64 ** 3 == 1_048_576 and 4 * 252 ** 3 == 64_012_032
    w = inputs.config(3, scale=0.01)
    assert w.N == 10_000 and abs(w.N / np.prod(w.box) - 3.0) < 1e-12 and w.dt == 0.02
    assert w.params["A"] == 25.0 and w.params["gamma"] == 4.5 and w.params["seed"] == 42


def test_polymer_recipe():
    w = inputs.config(4, scale=0.002)                                    # 40 chains x 64
    assert w.N == 40 * 64 and w.bonds.shape == (40 * 63, 2)
    d = w.pos[w.bonds[:, 0]] - w.pos[w.bonds[:, 1]]
    d -= w.box * np.rint(d / w.box)
    assert np.abs(np.sqrt((d * d).sum(1)) - 0.97).max() < 1e-12          # bond step 0.97
    assert np.all(w.bonds[:, 1] == w.bonds[:, 0] + 1)
    assert not np.any(w.bonds[:, 0] % 64 == 63)                          # no bond across chains
