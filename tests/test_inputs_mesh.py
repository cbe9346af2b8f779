"""The input generators' meshes obey the identities the method relies on; CPU only."""
import numpy as np
import pytest

from paper_2404_17630_b200.inputs import mesh as M


def _closure(m):
    C = m.ncell
    cl = np.zeros((3, C)); sa = np.zeros(C)
    ok = m.right >= 0
    for a in range(3):
        np.add.at(cl[a], m.left, m.area * m.normal[a])
        np.add.at(cl[a], m.right[ok], -(m.area * m.normal[a])[ok])
    np.add.at(sa, m.left, m.area); np.add.at(sa, m.right[ok], m.area[ok])
    return np.max(np.linalg.norm(cl, axis=0) / sa)


@pytest.mark.parametrize("periodic", [True, False])
def test_staggered_grid_is_a_body_centred_voronoi_mesh(periodic):
    """the "2 x N^3 staggered grid" = two interleaved cubic lattices; the Voronoi cell of
    a body-centred lattice point is a truncated octahedron with 14 faces (8 hexagons to the other lattice,
    6 squares to its own)."""
    n, box = 6, 2.0
    m = M.voronoi(n, box, 0.02, 3, periodic, stagger=True)
    assert m.ncell == 2 * n ** 3
    assert m.volume.sum() == pytest.approx(box ** 3, rel=1e-12)
    assert _closure(m) < 1e-12
    per_cell = np.bincount(m.left, minlength=m.ncell) + np.bincount(m.right[m.right >= 0], minlength=m.ncell)
    if periodic:
        assert np.all(per_cell == 14) and np.all(m.right >= 0)
        sub = np.arange(m.ncell) // n ** 3                       # 8 of the 14 neighbours sit on the other lattice
        cross = sub[m.left] != sub[m.right]
        assert cross.sum() * 2 == 8 * m.ncell
        assert m.volume == pytest.approx(np.full(m.ncell, box ** 3 / m.ncell), rel=0.2)
    else:
        assert (m.right < 0).sum() > 0 and per_cell.max() <= 15
    # sum_f A (c_f - s_i).(+-n) = 3 V_i  (divergence theorem on every closed cell)
    acc = np.zeros(m.ncell)
    r = m.fcentroid - m.centroid[:, m.left]
    np.add.at(acc, m.left, m.area * (r * m.normal).sum(0))
    ok = m.right >= 0
    d = m.fcentroid[:, ok] - m.centroid[:, m.right[ok]]
    for a in range(3):
        if periodic:
            d[a] -= box * np.rint(d[a] / box)
    np.add.at(acc, m.right[ok], -(m.area[ok] * (d * m.normal[:, ok]).sum(0)))
    assert np.allclose(acc, 3.0 * m.volume, rtol=1e-10)


def test_jittered_lattice_mesh_identities():
    m = M.voronoi(7, 1.0, 0.3, 11, True)
    assert m.volume.sum() == pytest.approx(1.0, rel=1e-12) and _closure(m) < 1e-12
    per_cell = np.bincount(m.left, minlength=m.ncell) + np.bincount(m.right, minlength=m.ncell)
    assert 13 < per_cell.mean() < 17
