"""Pins of oracle/fem.py (the CPU oracle of SURVEY.md 8(f)-4) against what linear elasticity and
linear algebra fix -- nothing here calls the CUDA path:

  * the Kuhn mesh tiles the volume (volumes add up, every interior face has exactly two tetrahedra);
  * K is symmetric positive semi-definite and its null space is exactly the six rigid-body modes;
  * patch test: a linear displacement field produces no force at interior nodes;
  * closed-form strain energies u^T K u = V * sigma:epsilon for uniaxial strain ((lambda + 2 mu) e^2), simple shear
    (mu g^2) and hydrostatic strain (3 (3 lambda + 2 mu) e^2), on an anisotropic mesh (catches swapped axes, a wrong
    Lame conversion, a missing factor in the shear rows);
  * the index form of the constant-strain element, K_ab = V (lambda g_a g_b^T + mu g_b g_a^T + mu (g_a . g_b) I);
  * H reproduces linear fields exactly and its rows sum to one;
  * the iteration of PAPER.md:258: a rigid translation is recovered exactly in one step and F stays 0; with K = 0 the
    step is the weighted least-squares solution (numpy.linalg.lstsq); the iterates converge monotonically to the
    interpolating solution (the fixed point H^T S H U = H^T S D); zero-confidence blocks have no influence.
"""
import itertools

import numpy as np
import pytest

from oracle import fem

E, NU = 3.0, 0.3
LAM, MU = fem.lame(E, NU)


def _mesh():
    return fem.mesh((13, 9, 11), (4, 2, 5))          # 4 x 5 x 3 nodes, anisotropic cells 4 x 2 x 5


def _dense_k(msh):
    return fem.stiffness(msh, E, NU).toarray()


def _tet_volume(x):
    return abs(np.linalg.det(np.hstack([np.ones((4, 1)), x]))) / 6.0


def test_lame_constants():
    lam, mu = fem.lame(1.0, 0.25)
    assert lam == pytest.approx(0.4) and mu == pytest.approx(0.4)        # E nu / ((1+nu)(1-2nu)), E / (2(1+nu))


def test_kuhn_mesh_tiles_the_volume():
    msh = _mesh()
    nnx, nny, nnz = msh["nodes_shape"]
    assert (nnx, nny, nnz) == (4, 5, 3) and len(msh["xyz"]) == 60 and len(msh["tets"]) == 6 * 3 * 4 * 2
    vols = np.asarray([_tet_volume(msh["xyz"][t]) for t in msh["tets"]])
    assert np.allclose(vols, 4 * 2 * 5 / 6.0) and vols.sum() == pytest.approx(12 * 8 * 10)
    faces = {}
    for t in msh["tets"]:
        for f in itertools.combinations(sorted(int(v) for v in t), 3):
            faces[f] = faces.get(f, 0) + 1
    assert set(faces.values()) == {1, 2}                                  # conforming: no face is shared by three
    xyz = msh["xyz"]
    lo, hi = xyz.min(axis=0), xyz.max(axis=0)
    for f, cnt in faces.items():                                          # a face seen once lies on the hull
        on_hull = any(np.all(xyz[list(f), a] == lo[a]) or np.all(xyz[list(f), a] == hi[a]) for a in range(3))
        assert (cnt == 1) == on_hull
    assert hi.tolist() == [12.0, 8.0, 10.0]                               # covers [0, n-1] on every axis


def test_stiffness_is_symmetric_psd_with_exactly_the_rigid_body_null_space():
    msh = _mesh()
    k = _dense_k(msh)
    assert np.allclose(k, k.T, atol=1e-12)
    x = msh["xyz"]
    modes = []
    for a in range(3):
        t = np.zeros_like(x); t[:, a] = 1.0
        modes.append(t.ravel())
    for w in np.eye(3):
        modes.append(np.cross(w, x).ravel())                              # infinitesimal rotation u = w x X
    for m in modes:
        assert np.max(np.abs(k @ m)) < 1e-10
    ev = np.linalg.eigvalsh(k)
    assert ev[0] > -1e-10 and np.sum(ev < 1e-9) == 6 and ev[6] > 1e-6


def test_patch_test_and_closed_form_strain_energies():
    msh = _mesh()
    k = _dense_k(msh)
    x = msh["xyz"]
    vol = 12.0 * 8.0 * 10.0
    nnx, nny, nnz = msh["nodes_shape"]
    interior = [(kk * nny + j) * nnx + i for kk in range(1, nnz - 1) for j in range(1, nny - 1) for i in range(1, nnx - 1)]
    a = np.asarray([[0.01, 0.02, -0.03], [0.00, -0.02, 0.05], [0.04, 0.01, 0.02]])
    f = (k @ (x @ a.T).ravel()).reshape(-1, 3)
    assert np.max(np.abs(f[interior])) < 1e-12                            # patch test
    e = 0.01
    for axis in range(3):                                                 # uniaxial strain along each axis
        u = np.zeros_like(x); u[:, axis] = e * x[:, axis]
        assert u.ravel() @ k @ u.ravel() == pytest.approx((LAM + 2 * MU) * e * e * vol, rel=1e-12)
    for i, j in ((0, 1), (1, 2), (2, 0), (1, 0)):                         # simple shear u_i = g x_j
        u = np.zeros_like(x); u[:, i] = e * x[:, j]
        assert u.ravel() @ k @ u.ravel() == pytest.approx(MU * e * e * vol, rel=1e-12)
    u = e * x
    assert u.ravel() @ k @ u.ravel() == pytest.approx(3 * (3 * LAM + 2 * MU) * e * e * vol, rel=1e-12)


def test_element_stiffness_equals_the_index_form():
    rng = np.random.default_rng(1)
    for _ in range(5):
        x = rng.uniform(0, 3, (4, 3))
        ke = fem.element_stiffness(x, E, NU)
        g = np.linalg.inv(np.hstack([np.ones((4, 1)), x]))[1:, :]         # gradients of the barycentric coordinates
        v = _tet_volume(x)
        for a in range(4):
            for b in range(4):
                want = v * (LAM * np.outer(g[:, a], g[:, b]) + MU * np.outer(g[:, b], g[:, a]) + MU * (g[:, a] @ g[:, b]) * np.eye(3))
                assert np.allclose(ke[3 * a:3 * a + 3, 3 * b:3 * b + 3], want, atol=1e-12)


def test_interpolation_reproduces_linear_fields():
    msh = _mesh()
    rng = np.random.default_rng(2)
    pts = np.vstack([rng.uniform(0, [12, 8, 10], (200, 3)), msh["xyz"][[0, 7, 59]], [[12, 8, 10], [4, 2, 5], [6, 3, 7.5], [2, 2, 2]]])
    h = fem.interpolation(msh, pts)
    assert np.allclose(np.asarray(h.sum(axis=1)).ravel(), 1.0)
    a = rng.normal(size=(3, 3)); b = rng.normal(size=3)
    nodal = msh["xyz"] @ a.T + b
    assert np.allclose((h @ nodal.ravel()).reshape(-1, 3), pts @ a.T + b, atol=1e-12)
    for p in pts:
        nodes, w = fem.locate(msh, p)
        assert np.all(w >= -1e-12) and w.sum() == pytest.approx(1.0) and np.allclose(w @ msh["xyz"][nodes], p)
    nodes, w = fem.locate(msh, msh["xyz"][7])                             # a node: weight one on itself
    assert nodes[np.argmax(w)] == 7 and w.max() == pytest.approx(1.0)


def _blocks_on(msh, rng, extra=80):
    """Integer block centres at every node plus some more: H then has full column rank."""
    pts = np.vstack([msh["xyz"], np.floor(rng.uniform(0, [12, 8, 10], (extra, 3)))])
    return pts.astype(np.int32)


def test_rigid_translation_is_recovered_exactly_and_the_force_stays_zero():
    msh = _mesh()
    rng = np.random.default_rng(3)
    c = _blocks_on(msh, rng)[::2]
    t = np.asarray([2.0, -1.0, 3.0])
    d = np.tile(t, (len(c), 1))
    r = fem.solve(msh, E, NU, c, d, rng.uniform(0.2, 1.0, len(c)), weight=0.7, n_iter=3)
    for u in r["iterates"]:
        assert np.allclose(u, t, atol=1e-9)
    assert np.max(np.abs(r["K"] @ r["U"].ravel())) < 1e-9


def test_without_stiffness_the_step_is_weighted_least_squares():
    msh = _mesh()
    rng = np.random.default_rng(4)
    c = _blocks_on(msh, rng)
    d = rng.normal(0, 2, (len(c), 3))
    ncc = rng.uniform(0.1, 1.0, len(c))
    r = fem.solve(msh, 0.0, NU, c, d, ncc, weight=2.5, n_iter=1)
    h = r["H"].toarray()
    sw = np.sqrt(np.repeat(2.5 * ncc, 3))
    want = np.linalg.lstsq(h * sw[:, None], d.ravel() * sw, rcond=None)[0]
    assert np.allclose(r["U"].ravel(), want, atol=1e-8)


def test_first_step_is_the_regularised_solution_and_iterates_converge_to_the_interpolating_one():
    msh = _mesh()
    rng = np.random.default_rng(5)
    c = _blocks_on(msh, rng)
    a = np.asarray([[0.02, 0.01, 0.0], [-0.01, 0.03, 0.02], [0.0, 0.01, -0.02]])
    u_lin = msh["xyz"] @ a.T + np.asarray([0.5, -0.25, 1.0])
    d = c.astype(np.float64) @ a.T + np.asarray([0.5, -0.25, 1.0])          # D = H U_lin exactly
    ncc = rng.uniform(0.3, 1.0, len(c))
    r = fem.solve(msh, E, NU, c, d, ncc, weight=5.0, n_iter=40)
    k, h, s = r["K"].toarray(), r["H"].toarray(), r["S"].toarray()
    first = np.linalg.solve(k + h.T @ s @ h, h.T @ s @ d.ravel())          # classical regularised least squares
    assert np.allclose(r["iterates"][0].ravel(), first, atol=1e-9)
    err = [np.max(np.abs(u - u_lin)) for u in r["iterates"]]
    assert err[0] > 1e-4                                                    # the mechanical forces do pull at first
    assert all(e1 <= e0 * (1 + 1e-12) + 1e-13 for e0, e1 in zip(err, err[1:]))
    assert err[-1] < 0.05 * err[0]                                            # "slowly cancel the influence of the mechanical forces"
    assert np.allclose(h.T @ s @ h @ u_lin.ravel(), h.T @ s @ d.ravel(), atol=1e-9)      # the fixed point


def test_blocks_without_confidence_have_no_influence():
    msh = _mesh()
    rng = np.random.default_rng(6)
    c = _blocks_on(msh, rng)
    d = rng.normal(0, 1, (len(c), 3))
    ncc = rng.uniform(0.2, 1.0, len(c))
    base = fem.solve(msh, E, NU, c, d, ncc, 1.0, 2)["U"]
    bad_c = np.vstack([c, [[3, 3, 3], [7, 5, 2], [1, 1, 9]]]).astype(np.int32)
    bad_d = np.vstack([d, [[100, 100, 100], [-50, 0, 7], [1, 2, 3]]])
    bad_n = np.concatenate([ncc, [-0.4, 0.0, np.nan]])
    assert np.allclose(fem.solve(msh, E, NU, bad_c, bad_d, bad_n, 1.0, 2)["U"], base, atol=1e-12)
    assert np.all(fem.confidence(np.asarray([0.5, -1.0, np.nan]), 2.0) == np.repeat([1.0, 0.0, 0.0], 3))


def test_dense_field_interpolates_the_nodal_displacements():
    msh = fem.mesh((7, 5, 6), (3, 2, 5))
    rng = np.random.default_rng(7)
    a = rng.normal(size=(3, 3)); b = rng.normal(size=3)
    u = msh["xyz"] @ a.T + b
    f = fem.dense_field(msh, u, (7, 5, 6))
    zz, yy, xx = np.meshgrid(np.arange(6), np.arange(5), np.arange(7), indexing="ij")
    p = np.stack([xx, yy, zz], axis=-1).astype(np.float64)
    assert np.allclose(np.moveaxis(f, 0, -1), p @ a.T + b, atol=1e-12)      # linear fields are reproduced at every voxel
    u2 = rng.normal(size=u.shape)
    f2 = fem.dense_field(msh, u2, (7, 5, 6))
    nnx, nny, nnz = msh["nodes_shape"]
    for n, (x, y, z) in enumerate(msh["xyz"].astype(int)):
        if x < 7 and y < 5 and z < 6:
            assert np.allclose(f2[:, z, y, x], u2[n])                       # at a node: that node's displacement
