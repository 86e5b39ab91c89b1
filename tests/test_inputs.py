"""Seeded input generators: determinism, SU(3) properties, documented RNG."""
import numpy as np

from paper_1311_5029_b200 import inputs as I


def test_splitmix64_reference_vector():
    # Public test vector of the splitmix64 generator: state 0 -> first output.
    assert int(I.splitmix64(np.array([0], dtype=np.uint64))[0]) == 0xE220A8397B1DCDAF


def test_normal_is_counter_based_and_standard():
    j = np.arange(200000)
    g = I.normal(7, 1, j)
    assert np.array_equal(g[1234:1300], I.normal(7, 1, j[1234:1300]))      # order independent
    assert abs(g.mean()) < 0.01 and abs(g.std() - 1) < 0.01
    assert not np.array_equal(g[:10], I.normal(8, 1, j[:10]))
    assert not np.array_equal(g[:10], I.normal(7, 2, j[:10]))


def _check_su3(U):
    eye = np.eye(3)
    assert np.abs(np.einsum("...ij,...kj->...ik", U, U.conj()) - eye).max() < 1e-13
    assert np.abs(np.linalg.det(U) - 1).max() < 1e-13


def test_links_are_su3_and_seeded():
    dims = (4, 3, 2, 2)
    U = I.near_identity_links(dims, 0.3, 1)
    _check_su3(U)
    assert np.array_equal(U, I.near_identity_links(dims, 0.3, 1))
    assert np.abs(U - np.eye(3)).max() < 1.5            # near identity
    H = I.haar_links(dims, 8)
    _check_su3(H)
    # Haar: <Re tr U>/3 ~ 0, mean plaquette ~ 0
    assert abs(np.trace(H, axis1=-2, axis2=-1).real.mean()) < 0.2
    assert abs(I.mean_plaquette(dims, H)) < 0.1
    assert I.tadpole_u0(I.mean_plaquette(dims, H)) == 1.0
    _check_su3(I.random_gauge_transform(dims, 4))


def test_plaquette_and_u0():
    dims = (4, 4, 4, 4)
    assert abs(I.mean_plaquette(dims, I.unit_links(dims)) - 1.0) < 1e-15
    U = I.near_identity_links(dims, 0.3, 1)
    pl = I.mean_plaquette(dims, U)
    assert 0.7 < pl < 0.9
    g = I.random_gauge_transform(dims, 4)
    assert abs(I.mean_plaquette(dims, I.gauge_transform_links(dims, U, g)) - pl) < 1e-13   # gauge invariant
    assert abs(I.tadpole_u0(pl) ** 4 - pl) < 1e-15


def test_site_indexing():
    dims = (4, 3, 2, 5)
    c = I.site_coords(dims)
    assert tuple(c[1]) == (1, 0, 0, 0) and tuple(c[4]) == (0, 1, 0, 0) and tuple(c[12]) == (0, 0, 1, 0)
    assert tuple(c[24]) == (0, 0, 0, 1)
    s = I.shifted_sites(dims, (1, 0, 0, 0))
    assert s[3] == 0 and s[0] == 1
    assert np.array_equal(I.shifted_sites(dims, (0, 0, 0, -1))[:24], np.arange(24) + 4 * 24)


def test_sources():
    dims = (2, 2, 2, 2)
    p = I.point_source(dims)
    assert p[0, 0] == 1 and np.abs(p).sum() == 1
    g = I.gaussian_spinor(dims, 2)
    assert g.shape == (16, 12) and np.array_equal(g, I.gaussian_spinor(dims, 2))
