"""Acceptance rules of BASELINE.json north_star, written once for every GPU parity test.

  * selected block set: bit-exact (same centres, same canonical order);
  * displacement: bit-exact, except blocks whose ORACLE top-two NCC values differ by < 1e-5 (counted);
  * NCC value: |gpu - oracle| <= 1e-4 absolute (for exempt blocks against the oracle NCC of the
    displacement the GPU chose, which is within 1e-5 of the oracle's best by construction).
"""
import numpy as np

NCC_TOL = 1e-4
TIE_BAND = 1e-5


def assert_select_parity(gpu_blocks, gpu_n, gpu_ncand, ora, gpu_var=None):
    assert gpu_ncand == ora["n_candidates"], (gpu_ncand, ora["n_candidates"])
    assert gpu_n == len(ora["centres"]), (gpu_n, len(ora["centres"]))
    g = np.asarray(gpu_blocks).reshape(-1, 3)
    assert np.array_equal(g, ora["centres"]), "selected block set / order differs from the oracle"
    if gpu_var is not None:
        v = np.asarray(gpu_var)
        # same two-pass, x-fastest, uncontracted double arithmetic on both sides: expect identical bits
        assert np.array_equal(v, ora["var"]), "max rel var diff %g" % np.max(np.abs(v - ora["var"]) / np.maximum(ora["var"], 1e-300))


def assert_match_parity(gpu_disp, gpu_ncc, ora, label=""):
    """Returns the number of exempt (photo-finish) blocks whose displacement differs."""
    gd = np.asarray(gpu_disp).reshape(-1, 3)
    gn = np.asarray(gpu_ncc, dtype=np.float64).reshape(-1)
    od, on, gap = ora["disp"], ora["ncc"], ora["gap"]
    assert gd.shape == od.shape and gn.shape == on.shape
    differ = np.any(gd != od, axis=1)
    exempt = gap < TIE_BAND
    bad = differ & ~exempt
    assert not bad.any(), "%s: %d displacement mismatches outside the 1e-5 tie band, first: block %d gpu %s oracle %s gap %g" % (
        label, int(bad.sum()), int(np.argmax(bad)), gd[np.argmax(bad)], od[np.argmax(bad)], gap[np.argmax(bad)])
    err = np.abs(gn - on)
    assert np.all(err <= NCC_TOL), "%s: max |dNCC| = %g at block %d" % (label, err.max(), int(err.argmax()))
    return int((differ & exempt).sum())
