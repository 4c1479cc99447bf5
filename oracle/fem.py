"""ORACLE (test infrastructure, CPU, float64) of the biomechanical regularisation that consumes the block-matching
result -- SURVEY.md section 8(f)-4.  Shares nothing with paper_2308_10868_b200/ (the CUDA path).  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / reference legs may import this package.

The paper (section 3): "Estimation of brain deformation is based on the finite element analysis (FEA)
using a linear elastic model ... We then iteratively seek such a position of the mesh vertices U that balances the
mechanical forces of the modeled tissue that resist deformation, with the external forces that correspond to the
displacements D estimated by block matching:

        F_i <= K U_i ,      U_{i+1} <= [K + H^T S H]^-1 [H^T S D + F_i]

K is the mechanical stiffness matrix, H is the interpolation matrix from the mesh vertices to the block matching
displacements, S is the matrix that captures the confidence in the block matching results.  F is the force that is
increasing between iterations to slowly cancel the influence of the mechanical forces."

The functions below follow that statement step by step with textbook ingredients, written out plainly (dense or scipy
sparse matrices, a library direct solve; no blocking, no matrix-free tricks):

  mesh(dims, spacing)          Q22  the mesh: the paper's mesher is out of scope, so a regular grid of nodes, every
                                    cell cut into the six Kuhn tetrahedra that share its main diagonal (conforming)
  element_stiffness(xyz, E, nu)      constant-strain tetrahedron, K_e = V B^T C B with the 6x12 strain-displacement
                                    matrix B and the 6x6 isotropic elasticity matrix C (Voigt notation)
  stiffness(mesh, E, nu)             assembly of K (3N x 3N, node-major: dof = 3*node + axis)
  interpolation(mesh, points)        H: the four barycentric weights of each point in its tetrahedron
  confidence(ncc, weight)      Q24  S = weight * diag(max(NCC, 0)) (one value per block, the same for its 3 axes)
  solve(...)                         the iteration above, U_0 = 0, a direct solve per iteration
  dense_field(mesh, U, dims)         the "dense deformation field that defines transformation for each point in the
                                    image space": U interpolated at every voxel

READINGS (Q22-Q25; the paper gives none of these): the mesh stand-in; E and nu are inputs (the
paper prints no material constants); S as above; displacements, node positions and U are in voxels.  Parity of these
readings is unpinned by the paper; the arithmetic is pinned by tests/test_fem_oracle_pins.py against closed forms of
linear elasticity (rigid-body null space, patch test, strain energies of uniaxial strain and simple shear),
weighted least squares (K = 0) and the fixed point of the iteration.
"""
from __future__ import annotations

import itertools
from typing import Dict, Sequence, Tuple

import numpy as np

# the six Kuhn tetrahedra of the unit cube: vertex 0, then one unit step along each axis in the order of a permutation
KUHN_PERMUTATIONS = list(itertools.permutations((0, 1, 2)))


def lame(young: float, poisson: float) -> Tuple[float, float]:
    """(lambda, mu) of an isotropic material."""
    lam = young * poisson / ((1.0 + poisson) * (1.0 - 2.0 * poisson))
    mu = young / (2.0 * (1.0 + poisson))
    return lam, mu


def mesh(dims: Sequence[int], spacing: Sequence[int]) -> Dict[str, np.ndarray]:
    """Regular tetrahedral grid mesh over a volume of dims = (nx, ny, nz) voxels (reading Q22).
    Nodes at (i*hx, j*hy, k*hz), enough of them to cover [0, n-1] per axis (at least 2); node index = (k*nny + j)*nnx + i.
    Returns nodes_shape (nnx, nny, nnz), xyz float64 [N][3] (voxels), tets int64 [T][4]."""
    nn = [max(2, -(-(int(dims[a]) - 1) // int(spacing[a])) + 1) for a in range(3)]
    nnx, nny, nnz = nn
    xyz = np.zeros((nnx * nny * nnz, 3), dtype=np.float64)
    for k in range(nnz):
        for j in range(nny):
            for i in range(nnx):
                xyz[(k * nny + j) * nnx + i] = (i * spacing[0], j * spacing[1], k * spacing[2])
    tets = []
    for k in range(nnz - 1):
        for j in range(nny - 1):
            for i in range(nnx - 1):
                for perm in KUHN_PERMUTATIONS:
                    c = [i, j, k]
                    verts = [(c[2] * nny + c[1]) * nnx + c[0]]
                    for axis in perm:
                        c[axis] += 1
                        verts.append((c[2] * nny + c[1]) * nnx + c[0])
                    tets.append(verts)
    return {"nodes_shape": (nnx, nny, nnz), "spacing": tuple(int(s) for s in spacing), "xyz": xyz,
            "tets": np.asarray(tets, dtype=np.int64)}


def elasticity_matrix(young: float, poisson: float) -> np.ndarray:
    """6x6 isotropic C in Voigt notation (xx, yy, zz, yz, xz, xy) with ENGINEERING shear strains."""
    lam, mu = lame(young, poisson)
    c = np.zeros((6, 6))
    c[:3, :3] = lam
    c[0, 0] = c[1, 1] = c[2, 2] = lam + 2.0 * mu
    c[3, 3] = c[4, 4] = c[5, 5] = mu
    return c


def element_stiffness(xyz4: np.ndarray, young: float, poisson: float) -> np.ndarray:
    """12x12 stiffness of the constant-strain tetrahedron with vertices xyz4 [4][3]: K_e = V B^T C B."""
    m = np.hstack([np.ones((4, 1)), np.asarray(xyz4, dtype=np.float64)])     # rows (1, x, y, z)
    vol = abs(np.linalg.det(m)) / 6.0
    grad = np.linalg.inv(m)[1:, :]                                          # grad[:, a] = gradient of shape function a
    b = np.zeros((6, 12))
    for a in range(4):
        gx, gy, gz = grad[:, a]
        b[0, 3 * a + 0] = gx
        b[1, 3 * a + 1] = gy
        b[2, 3 * a + 2] = gz
        b[3, 3 * a + 1] = gz; b[3, 3 * a + 2] = gy                          # gamma_yz
        b[4, 3 * a + 0] = gz; b[4, 3 * a + 2] = gx                          # gamma_xz
        b[5, 3 * a + 0] = gy; b[5, 3 * a + 1] = gx                          # gamma_xy
    return vol * b.T @ elasticity_matrix(young, poisson) @ b


def stiffness(msh, young: float, poisson: float):
    """K as a scipy CSR matrix (3N x 3N)."""
    from scipy import sparse
    n = len(msh["xyz"])
    rows, cols, vals = [], [], []
    for tet in msh["tets"]:
        ke = element_stiffness(msh["xyz"][tet], young, poisson)
        dof = np.asarray([3 * v + a for v in tet for a in range(3)])
        rows.append(np.repeat(dof, 12))
        cols.append(np.tile(dof, 12))
        vals.append(ke.ravel())
    k = sparse.coo_matrix((np.concatenate(vals), (np.concatenate(rows), np.concatenate(cols))), shape=(3 * n, 3 * n))
    return k.tocsr()


def locate(msh, point) -> Tuple[np.ndarray, np.ndarray]:
    """(node indices [4], barycentric weights [4]) of `point` (voxels) in its Kuhn tetrahedron.  Points on or beyond
    the last node plane belong to the last cell (weights may then leave [0, 1]: linear extrapolation)."""
    nnx, nny, nnz = msh["nodes_shape"]
    h = msh["spacing"]
    cell, loc = [], []
    for a, nn in enumerate((nnx, nny, nnz)):
        c = int(np.floor(point[a] / h[a]))
        c = min(max(c, 0), nn - 2)
        cell.append(c)
        loc.append(point[a] / h[a] - c)
    # the simplex whose permutation sorts the local coordinates in descending order (ties: lower axis first)
    perm = sorted(range(3), key=lambda a: (-loc[a], a))
    c = list(cell)
    nodes = [(c[2] * nny + c[1]) * nnx + c[0]]
    for axis in perm:
        c[axis] += 1
        nodes.append((c[2] * nny + c[1]) * nnx + c[0])
    s = [loc[a] for a in perm]
    w = [1.0 - s[0], s[0] - s[1], s[1] - s[2], s[2]]
    return np.asarray(nodes, dtype=np.int64), np.asarray(w, dtype=np.float64)


def interpolation(msh, points: np.ndarray):
    """H as a scipy CSR matrix (3P x 3N): row 3p+a interpolates axis a of the nodal field at point p."""
    from scipy import sparse
    n = len(msh["xyz"])
    rows, cols, vals = [], [], []
    for p, pt in enumerate(np.asarray(points, dtype=np.float64)):
        nodes, w = locate(msh, pt)
        for a in range(3):
            for v, wv in zip(nodes, w):
                rows.append(3 * p + a)
                cols.append(3 * int(v) + a)
                vals.append(wv)
    return sparse.coo_matrix((vals, (rows, cols)), shape=(3 * len(points), 3 * n)).tocsr()


def confidence(ncc: np.ndarray, weight: float) -> np.ndarray:
    """Diagonal of S (length 3P): weight * max(NCC, 0) per block (NaN counts as 0), repeated for the three axes (Q24)."""
    s = np.where(np.nan_to_num(np.asarray(ncc, dtype=np.float64), nan=0.0) > 0.0, np.nan_to_num(np.asarray(ncc, dtype=np.float64), nan=0.0), 0.0)
    return np.repeat(weight * s, 3)


def solve(msh, young: float, poisson: float, centres: np.ndarray, disp: np.ndarray, ncc: np.ndarray, weight: float,
          n_iter: int) -> Dict[str, np.ndarray]:
    """U_0 = 0; F_i = K U_i; U_{i+1} = [K + H^T S H]^-1 [H^T S D + F_i], i = 0 .. n_iter-1.
    centres int [P][3] (voxels), disp [P][3] (voxels), ncc [P].  Returns U [N][3] and the list of iterates."""
    from scipy import sparse
    from scipy.sparse.linalg import spsolve
    k = stiffness(msh, young, poisson)
    h = interpolation(msh, np.asarray(centres, dtype=np.float64))
    s = sparse.diags(confidence(ncc, weight))
    d = np.asarray(disp, dtype=np.float64).reshape(-1)
    a = (k + h.T @ s @ h).tocsc()
    rhs0 = h.T @ (s @ d)
    u = np.zeros(3 * len(msh["xyz"]))
    iterates = []
    for _ in range(int(n_iter)):
        f = k @ u
        u = spsolve(a, rhs0 + f)
        iterates.append(u.reshape(-1, 3).copy())
    return {"U": u.reshape(-1, 3), "iterates": iterates, "K": k, "H": h, "S": s}


def dense_field(msh, u: np.ndarray, dims: Sequence[int]) -> np.ndarray:
    """float64 [3][nz][ny][nx]: the nodal displacements interpolated at every voxel centre."""
    nx, ny, nz = dims
    out = np.zeros((3, nz, ny, nx), dtype=np.float64)
    u = np.asarray(u, dtype=np.float64).reshape(-1, 3)
    for z in range(nz):
        for y in range(ny):
            for x in range(nx):
                nodes, w = locate(msh, (float(x), float(y), float(z)))
                out[:, z, y, x] = w @ u[nodes]
    return out
