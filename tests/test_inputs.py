"""Seeded input generators (fmm_inputs): RNG test vector, Lane-Emden constants, cell model."""
import numpy as np

import fmm_inputs as fi
from helpers import moments_of_points


def test_splitmix64_reference_vector():
    # first outputs of the public-domain SplitMix64 generator for seed 1234567
    ref = [6457827717110365317, 3203168211198807973, 9817491932198370423, 4593380528125082431,
           16408922859458223821]
    assert fi.splitmix64(1234567, 5).tolist() == ref
    assert fi.splitmix64(1234567, 2, offset=3).tolist() == ref[3:5]
    u = fi.uniform01(42, 1000)
    assert (u >= 0).all() and (u < 1).all() and abs(u.mean() - 0.5) < 0.05


def test_lane_emden_n15_constants():
    """Textbook values for n = 3/2: xi_1 = 3.65375, -xi_1^2 theta'(xi_1) = 2.71406."""
    xs, ths, xi1 = fi.lane_emden()
    assert abs(xi1 - 3.65375) < 1e-4
    # mass integral: int_0^xi1 theta^1.5 xi^2 dxi = -xi1^2 theta'(xi1)
    integ = np.trapezoid(np.maximum(ths, 0) ** 1.5 * xs ** 2, xs)
    assert abs(integ - 2.71406) < 1e-4
    w = fi.config2(ncell=32)
    mass = 4 * np.pi * (0.4 / xi1) ** 3 * integ
    assert abs(w.moments[0].sum() - mass) / mass < 2e-3
    assert w.moments[0].min() >= fi.FLOOR * w.h ** 3 * 0.999


def test_config1_cell_model():
    w = fi.config1()
    assert w.n == (24, 24, 24) and w.out_lo == (8, 8, 8) and w.out_hi == (16, 16, 16)
    assert w.moments.shape == (20, 24, 24, 24) and w.com_off.shape == (3, 24, 24, 24)
    rho = w.moments[0] / w.h ** 3
    assert rho.min() >= 0.5 - 1e-12 and rho.max() <= 1.5 + 1e-12
    assert np.abs(w.com_off).max() <= 0.1 * w.h
    assert np.abs(w.moments[1:4]).max() < 1e-18          # centre-of-mass expansion: dipole = round-off
    assert (w.child_mass > 0).all()
    # moments of one cell recomputed from its children about its centre of mass
    k, j, i = 3, 17, 9
    y = np.array([(np.array([i, j, k]) + 0.5) * w.h + fi.CHILD_SIGNS[c] * 0.25 * w.h for c in range(8)])
    z = (np.array([i, j, k]) + 0.5) * w.h + w.com_off[:, k, j, i]
    ref = moments_of_points(w.child_mass[:, k, j, i], y, z)
    np.testing.assert_allclose(w.moments[:, k, j, i], ref, rtol=0, atol=1e-13 * np.abs(ref).max())
    # determinism
    w2 = fi.config1()
    assert np.array_equal(w.moments, w2.moments) and np.array_equal(w.com_off, w2.com_off)


def test_binary_mass_ratio_and_noise():
    w = fi.config3(ncell=64)
    m = w.moments[0]
    left, right = m[:, :, :32].sum(), m[:, :, 32:].sum()
    assert abs(right / left - 0.7) < 0.02
    w5 = fi.config5(ncell=32)
    w5b = fi._uniform_field("x", fi.BINARY, 32, 0.5, 1, None)
    ratio = w5.moments[0] / w5b.moments[0]
    assert np.abs(ratio - 1).max() <= 1.0001e-8 and np.abs(ratio - 1).max() > 1e-9
    w4 = fi.config4(ncell=32)
    assert w4.kind == "monopole" and w4.moments.shape == (1, 32, 32, 32) and w4.com_off is None


def test_uniform_sphere_of_section_3_4():
    """Radius 0.25, total mass 1, ambient 1e-10 of the sphere's density (L452); the analytic potential is continuous at
    the surface and -M/r outside."""
    h, mass, phi, r = fi.uniform_sphere(32)
    assert h == 1.0 / 32 and mass.shape == (32, 32, 32)
    assert abs(mass.sum() - 1.0) < 1e-14
    inside = r < 0.25
    assert np.isclose(mass[~inside].max() / mass[inside].min(), 1e-10, rtol=1e-12)
    assert abs(inside.sum() * h ** 3 / (4.0 / 3.0 * np.pi * 0.25 ** 3) - 1.0) < 0.03      # rasterised volume
    assert np.allclose(phi[~inside], -1.0 / r[~inside])
    assert np.isclose(-(3 * 0.0625 - 0.25 ** 2) / (2 * 0.25 ** 3), -1.0 / 0.25)           # continuity at r = R
    assert phi.min() > -1.5 / 0.25 - 1e-12                                                # centre value -3M/2R
