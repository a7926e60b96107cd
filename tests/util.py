"""Error metric of DESIGN.md R10 and small helpers shared by the tests."""
import numpy as np

TOL_ACC = 1.0e-5    # BASELINE.json north_star: max per-particle relative error, acc and pot
TOL_POT = 1.0e-5
TOL_JRK = 1.0e-4    # ... and jerk


def rel_err_vec(got, ref, floor=None):
    """Per-particle ||got - ref||_2 / ||ref||_2 for (3, n) arrays.  Where ||ref|| is below `floor`
    (an exactly symmetric case), the error is measured against the floor instead."""
    num = np.sqrt(((got - ref) ** 2).sum(0))
    den = np.sqrt((ref ** 2).sum(0))
    if floor is not None:
        den = np.maximum(den, floor)
    return num / den


def rel_err_scalar(got, ref):
    return np.abs(got - ref) / np.abs(ref)


def check_parity(got, ref, scale=1.0):
    """got/ref = (acc, jrk, pot); returns (e_acc, e_jrk, e_pot) maxima and asserts the north_star
    tolerances (times `scale`)."""
    ea = rel_err_vec(got[0], ref[0]).max() if ref[2].size else 0.0
    ej = rel_err_vec(got[1], ref[1]).max() if ref[2].size else 0.0
    ep = rel_err_scalar(got[2], ref[2]).max() if ref[2].size else 0.0
    assert ea <= TOL_ACC * scale, ("acc", ea)
    assert ej <= TOL_JRK * scale, ("jerk", ej)
    assert ep <= TOL_POT * scale, ("pot", ep)
    return ea, ej, ep
