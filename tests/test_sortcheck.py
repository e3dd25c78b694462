"""tests/sortcheck.py (the validity check of the exported order under the cell order, reading R22) accepts what it
should and rejects a wrong order: the checker itself is pinned, on the CPU."""
import numpy as np
import pytest

import oracle
from sortcheck import check_perm
from paper_2412_08265_b200 import synth


def case():
    w = synth.make_workload("tiny", n=5000)
    t = w.telescope
    key, _ = oracle.rotate_bin(w.particles.pos, w.particles.vel, w.rotation, t.n_x, t.n_y, t.spaxel_size)
    operm, oseg = oracle.sort(key, t.n_spaxels)
    ia, iz, _, _ = oracle.ssp_cells(w.particles.log_age, w.particles.log_z, w.ssp.log_age_axis, w.ssp.log_z_axis)
    cell = ia.astype(np.int64) * w.ssp.log_z_axis.size + iz
    cell = np.where(key < t.n_spaxels, cell, 0)
    cperm = np.lexsort((np.arange(key.size), cell, key)).astype(np.int32)      # (key, cell, index)
    return w, t, operm, oseg, cperm


def test_accepts_the_two_valid_orders():
    w, t, operm, oseg, cperm = case()
    args = (w.particles, w.ssp, t.n_spaxels)
    assert check_perm(operm, operm, oseg, *args, False) == "stable"
    assert check_perm(operm, operm, oseg, *args, None) == "stable"
    assert check_perm(cperm, operm, oseg, *args, True) == "cell"
    assert check_perm(cperm, operm, oseg, *args, None) == "cell"
    assert not np.array_equal(cperm, operm)


def test_rejects_wrong_orders():
    w, t, operm, oseg, cperm = case()
    args = (w.particles, w.ssp, t.n_spaxels)
    with pytest.raises(AssertionError):
        check_perm(cperm, operm, oseg, *args, False)                           # cell order where the stable one is required
    with pytest.raises(AssertionError):
        check_perm(operm, operm, oseg, *args, True)                            # and the other way round
    s = int(np.argmax(np.diff(oseg)[:-1]))                                     # the fullest spaxel
    a, b = int(oseg[s]), int(oseg[s + 1])
    swapped = cperm.copy()
    swapped[[a, b - 1]] = swapped[[b - 1, a]]                                  # same particles, not ordered by cell
    with pytest.raises(AssertionError):
        check_perm(swapped, operm, oseg, *args, None)
    moved = cperm.copy()
    moved[[a, int(oseg[s + 1])]] = moved[[int(oseg[s + 1]), a]]                # a particle in the wrong segment
    with pytest.raises(AssertionError):
        check_perm(moved, operm, oseg, *args, None)
