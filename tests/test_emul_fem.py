"""CPU tests (-m "not gpu") of the FEM kernels' LOGIC (paper_2308_10868_b200/csrc/nrr_fem.cu compiled against the
fiber emulation, tests/cuda_emul) against the oracle (oracle/fem.py): stencil stiffness from the cell table, FP64
scatter of H^T S H and H^T S D, the preconditioned conjugate gradients with device-side alpha / beta / convergence
flag, the F / U iteration of PAPER.md:258, the dense field.  The same comparisons run on the GPU in
tests/test_gpu_parity.py::test_fem_*."""
import numpy as np
import pytest

import _emul
from oracle import fem as ofem


def _case(dims, spacing, n_blocks, seed, amp=3):
    rng = np.random.default_rng(seed)
    msh = ofem.mesh(dims, spacing)
    nodes_in = msh["xyz"][np.all(msh["xyz"] < np.asarray(dims), axis=1)]
    extra = np.floor(rng.uniform(0, np.asarray(dims) - 1e-9, (n_blocks, 3)))
    blocks = np.vstack([nodes_in, extra]).astype(np.int32)
    disp = rng.integers(-amp, amp + 1, blocks.shape).astype(np.int32)
    ncc = rng.uniform(-0.2, 1.0, len(blocks)).astype(np.float32)
    ncc[::17] = np.nan
    return msh, blocks, disp, ncc


@pytest.mark.parametrize("dims,spacing,young,poisson,weight,n_iter", [
    ((13, 9, 11), (4, 2, 5), 3.0, 0.30, 1.0, 1),          # anisotropic cells, the classical regularised solution
    ((13, 9, 11), (4, 4, 5), 3.0, 0.45, 0.5, 2),          # nearly incompressible, two F / U iterations
    ((20, 20, 12), (5, 5, 5), 1.0, 0.10, 10.0, 2),
    ((9, 9, 9), (16, 16, 16), 2.0, 0.2, 1.0, 1),          # one cell: spacing beyond the volume
])
def test_emulated_fem_solve_matches_the_oracle(dims, spacing, young, poisson, weight, n_iter):
    msh, blocks, disp, ncc = _case(dims, spacing, 150, 11)
    want = ofem.solve(msh, young, poisson, blocks, disp, ncc, weight, n_iter)["U"]
    f = _emul.Fem(dims, spacing, young, poisson)
    assert f.nodes == msh["nodes_shape"] and f.n_nodes == len(msh["xyz"])
    got, iters, _ = f.solve(blocks, disp, ncc, weight, n_iter)
    assert iters > 0 and np.all(np.isfinite(got))
    assert np.max(np.abs(got - want)) <= 1e-6 * max(1.0, np.max(np.abs(want))), np.max(np.abs(got - want))
    # dense field: every voxel against the oracle's interpolation (fp32 output)
    field = f.dense_field(got)
    ref = ofem.dense_field(msh, got, dims)
    assert np.max(np.abs(field - ref)) <= 2e-6 * max(1.0, np.max(np.abs(ref)))
    f.destroy()


def test_emulated_fem_rigid_translation_and_empty_input():
    dims, spacing = (13, 9, 11), (4, 4, 5)
    msh, blocks, _, ncc = _case(dims, spacing, 60, 5)
    ncc = np.abs(np.nan_to_num(ncc, nan=0.5)) + 0.1
    disp = np.tile(np.asarray([2, -1, 3], np.int32), (len(blocks), 1))
    f = _emul.Fem(dims, spacing, 5.0, 0.4)
    u, iters, _ = f.solve(blocks, disp, ncc, 0.7, 2)
    assert np.allclose(u, [2.0, -1.0, 3.0], atol=1e-8)          # K annihilates rigid translations: recovered exactly
    u0, it0, _ = f.solve(blocks[:0], disp[:0], ncc[:0], 1.0, 2)
    assert np.all(u0 == 0.0) and it0 == 0                        # nothing to fit: U = 0, no CG iteration
    uz, _, _ = f.solve(blocks, disp, np.zeros(len(blocks), np.float32) - 1.0, 1.0, 1)
    assert np.all(uz == 0.0)                                     # no block with positive confidence
    f.destroy()


def test_emulated_fem_reports_non_convergence():
    dims, spacing = (13, 9, 11), (4, 2, 5)
    msh, blocks, disp, ncc = _case(dims, spacing, 100, 3)
    f = _emul.Fem(dims, spacing, 3.0, 0.3)
    u, iters, rc = f.solve(blocks, disp, ncc, 1.0, 1, tol=1e-13, max_cg=3, allow_noconv=True)
    assert rc == -13 and iters == 3 and np.all(np.isfinite(u))
    u2, iters2, rc2 = f.solve(blocks, disp, ncc, 1.0, 1)         # the model is reusable afterwards
    assert rc2 == 0 and iters2 > 3
    f.destroy()
