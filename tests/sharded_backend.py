"""Compute backend for the CPU tests of paper_2412_08265_b200/sharded.py: the fp64 oracle stands in for the CUDA library,
so that the HOST logic (routing, partition, all-to-all, halo exchange) runs where there is no GPU.  Test code only."""
import dataclasses

import numpy as np
import torch

import oracle
from paper_2412_08265_b200 import synth


def particles_of(records):
    r = records.cpu().numpy()
    return synth.Particles(np.ascontiguousarray(r[:, 0:3]), np.ascontiguousarray(r[:, 3:6]), np.ascontiguousarray(r[:, 6]),
                           np.ascontiguousarray(r[:, 7]), np.ascontiguousarray(r[:, 8]))


class OracleBackend:
    dtype = torch.float64

    def bin(self, records, tel, R):
        p = particles_of(records)
        key, _ = oracle.rotate_bin(p.pos, p.vel, R, tel.n_x, tel.n_y, tel.spaxel_size)
        return torch.from_numpy(key)

    def upload_flux(self, ssp):
        return None

    def build_rows(self, records, R, ssp, flux_dev, tel, x0, x1, out, mirror_lo=None, mirror_hi=None, mirror_rows=0):
        n_y, n_c = tel.n_y, tel.n_channels
        sel = np.arange(x0 * n_y, x1 * n_y, dtype=np.int32)
        if sel.size:
            cube = oracle.build_cube(particles_of(records), R, ssp, tel, sel=sel)
            out.copy_(torch.from_numpy(cube.reshape(x1 - x0, n_y, n_c)))
        if mirror_lo is not None:                              # the fused halo write of rubix_build_cube_mirrored
            mirror_lo.copy_(out[:mirror_rows])
        if mirror_hi is not None:
            mirror_hi.copy_(out[out.shape[0] - mirror_rows:])
        return None

    def convolve_rows(self, rows, tel):
        sub = dataclasses.replace(tel, n_x=int(rows.shape[0]))
        sk = oracle.psf_sigma_k(sub)
        return torch.from_numpy(oracle.convolve(rows.numpy(), sub.psf_size, sub.psf_sigma, sub.lsf_size, sub.lsf_sigma, sk))
