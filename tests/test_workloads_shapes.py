"""Host-side checks of the shape / layout generators (workloads.py): the generatrix quadratures reproduce the closed-form
surface areas and volumes of their bodies, and the paper-like lens layout respects the method's non-overlap assumption."""
import numpy as np

from paper_2107_09879_b200 import workloads as W


def area_volume(gen):
    th, r, dr, w = gen
    area = 2.0 * np.pi * np.sum(w * r * np.sin(th) * np.sqrt(r * r + dr * dr))
    volume = 2.0 * np.pi / 3.0 * np.sum(w * r ** 3 * np.sin(th))
    return area, volume


def test_generatrix_quadratures_reproduce_area_and_volume():
    a, v = area_volume(W.generatrix_sphere(0.2, 48))
    assert abs(a - 4 * np.pi * 0.04) < 1e-13 and abs(v - 4 * np.pi / 3 * 0.008) < 1e-13
    a, v = area_volume(W.generatrix_sphere(0.2, 64, offset=0.07))                     # same sphere seen off-centre
    assert abs(a - 4 * np.pi * 0.04) < 1e-12 and abs(v - 4 * np.pi / 3 * 0.008) < 1e-12
    rad, h = 0.15, 0.4
    a, v = area_volume(W.generatrix_cylinder(rad, h, 32))
    assert abs(a - (2 * np.pi * rad * h + 2 * np.pi * rad ** 2)) < 1e-12 and abs(v - np.pi * rad ** 2 * h) < 1e-12
    ax, cz = 0.15, 0.22
    e = np.sqrt(1 - ax ** 2 / cz ** 2)
    a, v = area_volume(W.generatrix_spheroid(ax, cz, 64))
    assert abs(a - 2 * np.pi * ax ** 2 * (1 + cz / (ax * e) * np.arcsin(e))) < 1e-11     # prolate spheroid
    assert abs(v - 4 * np.pi / 3 * ax ** 2 * cz) < 1e-12


def test_generatrix_derivative_matches_the_radius_function():
    for gen_fn in (lambda n: W.generatrix_sphere(0.2, n, offset=0.05), lambda n: W.generatrix_spheroid(0.15, 0.22, n)):
        th, r, dr, _ = gen_fn(200)
        order = np.argsort(th)
        num = np.gradient(r[order], th[order], edge_order=2)
        assert np.abs(num[5:-5] - dr[order][5:-5]).max() < 1e-3


def test_paper_lens_layout():
    w = W.paper_lens(56)
    assert w["pos"].shape == (3136, 3) and np.all(w["pos"][:, 2] == 0.0)
    assert w["type_of"].min() >= 0 and w["type_of"].max() < len(w["radii"]) and len(np.unique(w["type_of"])) > 16
    r_enc = np.sqrt(w["radii"].max() ** 2 + (0.5 * w["height"]) ** 2)
    assert 2.0 * r_enc < w["pitch"]                       # enclosing spheres do not intersect
    assert abs(56 * w["pitch"] * 1.55 - 60.0) < 0.2      # 60 um aperture
