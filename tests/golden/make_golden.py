"""Writes the stored expected values under tests/golden/.  Calls ONLY the seeded generator
(paper_2412_08265_b200.synth) and the oracle (oracle/); never the CUDA path.

  python tests/golden/make_golden.py

synth_sha256.json   SHA-256 of every input array of the tiny and small workloads: detects drift
                    of the generator ("SHA-256 of each array is recorded").
oracle_tiny.json    a few scalars of the oracle's tiny cube (config 0): per-spaxel counts, total
                    flux, the brightest voxel, three sample voxels; detects drift of the oracle.
The paper prints no worked numeric example (PAPER.md has no tables), so there is no
paper-sourced fixture; the only paper/SURVEY-quoted constant, sigma(FWHM=3) = 1.273983, is
asserted in tests/test_oracle_convolve.py.
"""
import json
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import oracle  # noqa: E402
from paper_2412_08265_b200 import synth  # noqa: E402


def main():
    hashes = {}
    for name in ("tiny", "small"):
        w = synth.make_workload(name)
        for f in ("pos", "vel", "mass", "log_age", "log_z"):
            hashes[f"{name}.particles.{f}"] = synth.sha256(getattr(w.particles, f))
        hashes[f"{name}.ssp.flux"] = synth.sha256(w.ssp.flux)
        hashes[f"{name}.ssp.log_age_axis"] = synth.sha256(w.ssp.log_age_axis)
        hashes[f"{name}.ssp.log_z_axis"] = synth.sha256(w.ssp.log_z_axis)
        hashes[f"{name}.rotation"] = synth.sha256(w.rotation)
    for name in ("medium", "contention"):
        hashes[f"{name}.euler_deg"] = [round(v, 9) for v in synth.euler_for(name)]
    with open(os.path.join(HERE, "synth_sha256.json"), "w") as f:
        json.dump(hashes, f, indent=1, sort_keys=True)

    w = synth.make_workload("tiny")
    t = w.telescope
    cube = oracle.forward(w.particles, w.rotation, w.ssp, t)
    key, _ = oracle.rotate_bin(w.particles.pos, w.particles.vel, w.rotation, t.n_x, t.n_y, t.spaxel_size)
    fix = {
        "n_in_fov": int((key < t.n_spaxels).sum()),
        "max_count": int(np.bincount(key)[:-1].max()),
        "total_flux": float(cube.sum()),
        "max_voxel": float(cube.max()),
        "argmax": [int(v) for v in np.unravel_index(cube.argmax(), cube.shape)],
        "voxels": {"8,8,100": float(cube[8, 8, 100]), "3,12,0": float(cube[3, 12, 0]),
                   "15,0,255": float(cube[15, 0, 255])},
    }
    with open(os.path.join(HERE, "oracle_tiny.json"), "w") as f:
        json.dump(fix, f, indent=1, sort_keys=True)


if __name__ == "__main__":
    main()
