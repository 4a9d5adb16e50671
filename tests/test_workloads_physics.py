"""Pins of the analytic input recipes of the paper's Section 4.1 (workloads.py) against what the paper prints."""
import os

import numpy as np

import workloads as wl

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "harris_roots.txt")


def test_harris_dispersion_vanishes_at_the_papers_roots():
    """Eq. 34 evaluated with the paper's fifty-point quadrature at the roots the paper prints (three digits): |eps| is
    1e-3 there and O(1) a short distance away in omega or k."""
    rows = np.loadtxt(GOLDEN)
    for k, wr, wi in rows:
        w = complex(wr, wi)
        at_root = abs(wl.harris_dispersion(w, k, 6, 10.0))
        assert at_root < 5e-3, (k, w, at_root)
        assert abs(wl.harris_dispersion(w + 0.15j, k, 6, 10.0)) > 50 * at_root
        assert abs(wl.harris_dispersion(w, k + 0.12, 6, 10.0)) > 50 * at_root


def test_ring_distribution_is_normalised_and_matches_config_ring():
    """Eq. 31 integrates to one (trapezoid on a fine grid; the integrand and all derivatives vanish at the box edge) and for
    j = 3 equals the config-2/3 recipe (reading C17: peak 0.03566)."""
    v = np.linspace(-12.0, 12.0, 1201)
    for j in (0, 3, 6):
        f = wl.ring_distribution(v, v, j)
        assert abs(f.sum() * (v[1] - v[0]) ** 2 - 1.0) < 1e-10
    f3 = wl.ring_f0(np.array([0.0]), v, v, 0.1, amp=0.0)[0]
    assert np.max(np.abs(f3 - wl.ring_distribution(v, v, 3))) < 1e-15
    assert abs(f3.max() - 0.03566) < 1e-5


def test_eigenmode_perturbation_structure():
    """Eq. 35-36: f1 has the wavenumber k in x (f1(x + pi/k) = -f1(x)), carries no net charge over a wavelength, and
    its velocity part is the (1/v) df0/dv envelope of Eq. 32 (zero on the ring maximum v_perp^2 = 2 j alpha^2)."""
    k_sim, kL, w = 0.0886, 0.886, 0.349j
    x = np.linspace(0.0, 2 * np.pi / k_sim, 17)[:-1]
    v = np.linspace(-8.5, 8.5, 69)
    f1 = wl.eigenmode_perturbation(x, v, v, k_sim, kL, w, 6)
    assert np.max(np.abs(f1[8:] + f1[:8])) < 1e-12 * np.max(np.abs(f1))
    assert abs(f1.sum()) < 1e-10 * np.abs(f1).sum()
    vr = np.sqrt(12.0)
    on_ring = wl.eigenmode_perturbation(x, np.array([vr, 0.0]), np.array([0.0, vr]), k_sim, kL, w, 6)
    assert abs(on_ring[0, 0, 0]) < 1e-14 and abs(on_ring[0, 1, 1]) < 1e-14
    assert np.all(np.isfinite(wl.eigenmode_perturbation(x, np.array([0.0]), np.array([0.0]), k_sim, kL, w, 6)))
