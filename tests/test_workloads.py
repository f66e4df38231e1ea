"""Seeded input generators against the check values of SURVEY.md §8(d) / P11 / P12."""
import json
import os

import numpy as np

from paper_2112_08264_b200 import workloads as w

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "p12_config0_trajectory.json")))


def test_mix_check_values():
    assert int(w.mix(0)) == int(GOLD["mix"]["0"], 16)
    assert int(w.mix(1)) == int(GOLD["mix"]["1"], 16)


def test_u01_check_values_and_range():
    got = w.u01(GOLD["seed"], np.arange(4))
    assert got.tolist() == GOLD["u01_ctr0_3"]
    big = w.u01(7, np.arange(100000))
    assert big.min() >= 0.0 and big.max() < 1.0
    assert abs(big.mean() - 0.5) < 5e-3


def test_config0_fields():
    rr, rb = w.CONFIGS[0].fields()
    assert rr[:3].tolist() == GOLD["rho_r_n0_2"]
    assert rb[:3].tolist() == GOLD["rho_b_n0_2"]
    assert abs(rr.sum() - GOLD["mass"][0]) < 1e-8
    assert abs(rb.sum() - GOLD["mass"][1]) < 1e-8
    assert np.all(np.abs(rr - 1.0) <= 0.01) and np.all(np.abs(rb - 1.0) <= 0.01)


def test_fields_chunking_is_invisible():
    a = w.mixture_fields(8, 4, 4, 99, chunk=7)
    b = w.mixture_fields(8, 4, 4, 99, chunk=1 << 20)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_single_sphere_counts():
    g = GOLD["geometry"]
    m = w.solid_mask_from_spheres(32, 32, 32, np.array([[16.0, 16.0, 16.0]]))
    assert int(m.sum()) == g["sphere_R5.5_on_node"]["solid"]
    m = w.solid_mask_from_spheres(32, 32, 32, np.array([[16.5, 16.5, 16.5]]))
    assert int(m.sum()) == g["sphere_R5.5_on_cell_centre"]["solid"]
    # brute force over every node, straight from the definition (reading S9)
    c = np.array([3.2, 30.9, 15.4])
    z, y, x = np.meshgrid(np.arange(32), np.arange(32), np.arange(32), indexing="ij")
    d2 = sum(np.minimum(np.abs(a - ci), 32 - np.abs(a - ci)) ** 2 for a, ci in ((x, c[0]), (y, c[1]), (z, c[2])))
    want = (d2 <= 30.25).astype(np.uint8).reshape(-1)
    assert np.array_equal(w.solid_mask_from_spheres(32, 32, 32, c[None]), want)


def test_config4_packing_pins():
    g = GOLD["geometry"]["config4"]
    cfg = w.CONFIGS[4]
    centres, drawn = w.sphere_centres(cfg.nx, cfg.ny, cfg.nz, cfg.sphere_seed, cfg.n_spheres)
    assert drawn == g["candidates"]
    assert np.allclose(centres[0], g["first_centre"], atol=5e-9)
    # non-overlap under the minimum image
    box = np.array([256.0] * 3)
    for i in (0, 17, 1999):
        d = np.abs(centres - centres[i])
        d = np.minimum(d, box - d)
        r = np.sqrt((d * d).sum(1))
        r[i] = 1e9
        assert r.min() >= 11.0
    mask = w.solid_mask_from_spheres(cfg.nx, cfg.ny, cfg.nz, centres)
    assert int(mask.sum()) == g["solid"]
