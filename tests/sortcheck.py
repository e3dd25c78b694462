"""Comparison of the exported sort artefacts with the oracle.

key and seg_off are unique and compared bit for bit.  perm is unique when it is the stable order by (key, index); with the
cell order (rubix_telescope.cell_order) the particles of a spaxel come ordered by (SSP cell, index) instead: the segments
must then hold the same particles as the oracle's (compared after sorting each segment), and the order inside a segment is
checked against the cells the ORACLE finds for the particles."""
import numpy as np

import oracle


def check_perm(perm, operm, oseg, particles, ssp, n_spaxels, cell_order):
    """cell_order: False = perm must be the stable order; True = must be the (key, cell, index) order;
    None = either of the two."""
    perm = np.asarray(perm).astype(np.int64)
    operm = np.asarray(operm).astype(np.int64)
    if cell_order is False or (cell_order is None and np.array_equal(perm, operm)):
        assert np.array_equal(perm, operm), "sort order differs"
        return "stable"
    seg_id = np.repeat(np.arange(oseg.size - 1), np.diff(oseg))
    assert seg_id.size == perm.size
    inside = np.lexsort((perm, seg_id))                        # ascending index inside every segment
    assert np.array_equal(perm[inside], operm), "a segment holds other particles than the oracle's"
    ia, iz, _, _ = oracle.ssp_cells(particles.log_age, particles.log_z, ssp.log_age_axis, ssp.log_z_axis)
    cell = (ia.astype(np.int64) * ssp.log_z_axis.size + iz)[perm]
    cell[seg_id >= n_spaxels] = 0                              # dropped particles: plain index order
    same = seg_id[1:] == seg_id[:-1]
    ordered = (cell[1:] > cell[:-1]) | ((cell[1:] == cell[:-1]) & (perm[1:] > perm[:-1]))
    assert ordered[same].all(), "order inside a spaxel is not (SSP cell, index)"
    return "cell"
