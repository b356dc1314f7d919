"""The seeded input generators (paper_2512_04447_b200/workloads.py) that feed both the oracle and the CUDA path:
determinism, column independence, and the geometric facts of the five configs stated in DESIGN.md section 4."""
import numpy as np

from paper_2512_04447_b200 import workloads as wl


def test_orbital_columns_are_seeded_per_column_and_block_y_matches():
    ng = 64
    a = wl.orbital_block(ng, [3, 5, 0], 9, 1)
    b = wl.orbital_block(ng, [0, 5], 9, 1)
    assert np.array_equal(a[2].numpy(), b[0].numpy()) and np.array_equal(a[1].numpy(), b[1].numpy())
    assert not np.array_equal(wl.orbital_block(ng, [0], 9, 2).numpy(), b[:1].numpy())          # another stream
    system = dict(m=3, n=(4, 4, 4), seed=9)
    Y = wl.block_y(system, device="cpu")
    for s in range(3):
        assert np.array_equal(Y[3 * s:3 * s + 3].numpy(), wl.orbital_block(ng, range(3), 9, s).numpy())
    v = Y.numpy().reshape(-1)
    assert abs(np.mean(np.abs(v) ** 2) - 1.0) < 0.2                                            # CN(0, 1)


def test_config_geometry_matches_the_stated_recipe():
    for cfg, natom, nproj in ((0, 2, 4), (1, 16, 4), (2, 216, 4), (3, 128, 9)):
        s = wl.make_system(cfg, with_vloc=False, check_margin=False)
        assert len(s["pos"]) == natom and len(s["species"][0]["l"]) == nproj
        assert np.all(s["pos"] >= 0) and np.all(s["pos"] < s["len"][0])
    d = wl.make_system(2, with_vloc=False, check_margin=False)
    h = d["len"][0] / d["n"][0]
    assert np.max(np.abs(d["pos"] / h - np.round(d["pos"] / h))) < 1e-9                        # diamond atoms sit on grid points
    w = wl.make_system(3, with_vloc=False, check_margin=False)
    D = w["species"][0]["D"]
    assert np.allclose(D, np.diag(np.diag(D))) and np.all(np.abs(np.diag(D)) <= 1.0)           # D = diag(U[-1, 1])
    assert np.array_equal(D, wl.make_system(3, with_vloc=False, check_margin=False)["species"][0]["D"])   # seeded
