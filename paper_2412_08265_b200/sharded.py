"""Spaxel-sharded forward model over several GPUs (the paper's multi-GPU runs).

The paper shards by particle with ``pmap`` and gathers partial cubes (scaling "not perfect", L66).  Here the DETECTOR is
sharded instead: after steps 1-2 every particle is sent to the rank that owns its detector row, so each rank reduces
whole spaxels locally and the cube is never exchanged -- only 36-byte particle records (one all-to-all) and the
(psf_size - 1) / 2 raw rows next to each boundary (one halo exchange with the two neighbours).

  1  rubix_bin_particles on the rank's slice of the particle arrays (keys in the geometry of the WHOLE detector)
  2  rows per detector row: local histogram, all-reduce (n_x integers)
  3  partition_rows: contiguous row ranges of about equal cost (particles + a fixed cost per row)
  4  all-to-all of the particle records, source order kept: ranks hold contiguous slices of the original arrays, so a
     rank receives its particles in ORIGINAL order and the stable (key, index) order of step 3 is the single-GPU one
  5  rubix_build_cube on the rank's row window (rubix_telescope.n_x_full / x_first) into a buffer with room for the halos
  6  halo exchange of raw rows with the neighbouring ranks -- or, where a rank can store into its neighbours' buffers
     (ranks of one process; peer-mapped memory), steps 5 + 6 FUSED: rubix_build_cube_mirrored lets the kernels that produce
     the boundary rows write them into the neighbours' halos as well, and the exchange shrinks to a barrier
  7  rubix_convolve_psf_lsf on rows + halos; the rank keeps its own rows of the final cube
Every spaxel is summed by one rank over the same particles in the same order and chunks as on one GPU, and the stencils see
the same neighbours, so the slabs equal the single-GPU cube bit for bit.

All arithmetic of the method runs in the library's kernels (through ``backend``); this module is host logic: routing,
partitioning and the two exchanges, written once for any communicator (``DistComm`` = torch.distributed, NCCL or gloo;
``ThreadComm`` = the ranks of one process, used to run the sharded path on a single GPU).  The default product backend is
``CudaBackend`` (the C ABI); tests pass their own.  No data-path collective beyond the three named above.
"""
from __future__ import annotations

import dataclasses
import threading

import numpy as np

RECORD_FLOATS = 9        # pos[3], vel[3], mass, log_age, log_z
CELL_AUTO_MEAN = 64      # rubix.h: RUBIX_CELL_ORDER_AUTO turns the cell order on from this many particles per spaxel ...
CELL_AUTO_MIN_N = 1_000_000   # ... and this many particles


# ------------------------------------------------------------------------------------------ partitioning
def partition_rows(row_counts, world: int, min_rows: int = 1, row_cost: float = 0.0) -> np.ndarray:
    """Boundaries b[0] = 0 <= ... <= b[world] = n_x of contiguous row ranges with about equal cost, where a row costs
    ``row_counts[x] + row_cost`` (its particles plus a fixed share for zero fill and the stencil passes).  Every rank
    gets at least ``min_rows`` rows (the halo exchange reaches one neighbour only).  Deterministic: the same on all ranks."""
    counts = np.asarray(row_counts, dtype=np.float64)
    n_x = counts.size
    if world < 1 or min_rows < 1:
        raise ValueError("world and min_rows must be >= 1")
    if n_x < world * min_rows:
        raise ValueError(f"{n_x} detector rows cannot give {world} ranks {min_rows} rows each")
    cost = counts + float(row_cost)
    prefix = np.concatenate([[0.0], np.cumsum(cost)])
    total = prefix[-1]
    bounds = np.zeros(world + 1, dtype=np.int64)
    bounds[world] = n_x
    for r in range(1, world):
        target = total * r / world
        b = int(np.searchsorted(prefix, target, side="left"))
        if b > 0 and abs(prefix[b - 1] - target) <= abs(prefix[min(b, n_x)] - target):
            b -= 1                                          # the nearer of the two candidate boundaries
        lo = bounds[r - 1] + min_rows                       # leave min_rows to this rank and to every later one
        hi = n_x - (world - r) * min_rows
        bounds[r] = min(max(b, lo), hi)
    return bounds


def owner_of_rows(rows, bounds):
    """Rank that owns each detector row (torch tensor in, torch tensor out)."""
    import torch
    inner = torch.as_tensor(np.asarray(bounds[1:-1]), device=rows.device, dtype=rows.dtype)
    return torch.bucketize(rows, inner, right=True)


# ------------------------------------------------------------------------------------------ communicators
class DistComm:
    """torch.distributed (NCCL on GPUs, gloo on CPU): point-to-point messages only, plus one all-reduce / all-gather."""

    def __init__(self):
        import torch.distributed as dist
        self.dist = dist
        self.rank, self.world = dist.get_rank(), dist.get_world_size()

    def all_reduce_sum(self, t):
        self.dist.all_reduce(t)
        return t

    def all_gather_counts(self, t):
        out = [t.new_zeros(t.shape) for _ in range(self.world)]
        self.dist.all_gather(out, t)
        return out

    def share(self, obj):
        """Ranks are separate processes: no rank can store into another rank's buffer through this communicator (peer
        pointers would need CUDA IPC handles), so the halo goes through `exchange`."""
        return None

    def barrier(self):
        self.dist.barrier()

    def exchange(self, sends: dict, recv_shapes: dict, like):
        """sends: {peer: tensor}; recv_shapes: {peer: shape}.  Returns {peer: tensor}."""
        import torch
        dist = self.dist
        recvs = {p: torch.empty(shape, dtype=like.dtype, device=like.device) for p, shape in recv_shapes.items()}
        ops = [dist.P2POp(dist.isend, t.contiguous(), p) for p, t in sorted(sends.items()) if t.numel()]
        ops += [dist.P2POp(dist.irecv, t, p) for p, t in sorted(recvs.items()) if t.numel()]
        if ops:
            for req in dist.batch_isend_irecv(ops):
                req.wait()
        return recvs


class ThreadComm:
    """The ranks of ONE process, one thread each (``run_threads``): messages go through a shared mailbox, collectives
    through a barrier.  The threads only ever block on the host, never inside a kernel."""

    class Shared:
        def __init__(self, world):
            self.world, self.barrier, self.box = world, threading.Barrier(world), {}

    def __init__(self, shared, rank):
        self.s, self.rank, self.world = shared, rank, shared.world

    def _gather(self, tag, value):
        self.s.box[(tag, self.rank)] = value
        self.s.barrier.wait()
        vals = [self.s.box[(tag, r)] for r in range(self.world)]
        self.s.barrier.wait()
        if self.rank == 0:
            for r in range(self.world):
                del self.s.box[(tag, r)]
        self.s.barrier.wait()
        return vals

    def all_reduce_sum(self, t):
        vals = self._gather("sum", t.clone())
        t.copy_(sum(vals[1:], vals[0].clone()))
        return t

    def all_gather_counts(self, t):
        return [v.clone() for v in self._gather("cnt", t.clone())]

    def share(self, obj):
        """The ranks live in one address space: every rank gets every rank's object (here: its raw-row buffer), so a
        rank's kernels can store straight into a neighbour's halo."""
        return self._gather("share", obj)

    def barrier(self):
        self._gather("bar", None)

    def exchange(self, sends: dict, recv_shapes: dict, like):
        import torch
        all_sends = self._gather("p2p", {p: t.clone() for p, t in sends.items()})
        out = {}
        for p, shape in recv_shapes.items():
            t = all_sends[p].get(self.rank)
            out[p] = t if t is not None else torch.empty(shape, dtype=like.dtype, device=like.device)
            assert tuple(out[p].shape) == tuple(shape)
        return out


def run_threads(world: int, fn):
    """Runs fn(comm) for ``world`` ThreadComm ranks and returns the list of results (exceptions re-raised)."""
    shared = ThreadComm.Shared(world)
    results, errors = [None] * world, []

    def work(r):
        try:
            results[r] = fn(ThreadComm(shared, r))
        except BaseException as exc:                        # noqa: BLE001 -- surfaced below; a broken rank releases the others
            errors.append(exc)
            shared.barrier.abort()

    threads = [threading.Thread(target=work, args=(r,)) for r in range(world)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    if errors:
        first = [e for e in errors if not isinstance(e, threading.BrokenBarrierError)]
        raise (first or errors)[0]
    return results


# ------------------------------------------------------------------------------------------ product backend
class CudaBackend:
    """Steps of the sharded path on the C ABI (librubix_b200.so).  No fallback: loading fails without the library."""

    def __init__(self, device="cuda:0"):
        import torch
        from . import binding
        binding.load()
        self.B, self.torch, self.device = binding, torch, torch.device(device)

    def bin(self, records, tel, R):
        B, torch = self.B, self.torch
        key = torch.empty(records.shape[0], dtype=torch.int32, device=self.device)
        pos, vel = records[:, 0:3].contiguous(), records[:, 3:6].contiguous()
        B.rubix_bin_particles(pos, vel, B.c_telescope(tel), R, key)
        return key

    def build_rows(self, records, R, ssp, flux_dev, tel, x0, x1, out, mirror_lo=None, mirror_hi=None, mirror_rows=0):
        """Raw cube rows x0 .. x1 - 1 of the whole detector ``tel`` from ``records`` into ``out`` [x1 - x0, n_y, n_c]; with
        mirrors, the first / last ``mirror_rows`` rows are also stored there by the producing kernels (the fused halo write)."""
        B, torch = self.B, self.torch
        sub = dataclasses.replace(tel, n_x=int(x1 - x0), n_x_full=int(tel.n_x), x_first=int(x0))
        cols = [records[:, 0:3].contiguous(), records[:, 3:6].contiguous()] + [records[:, c].contiguous() for c in (6, 7, 8)]
        cp, cs, ct = B.c_particles(*cols), B.c_ssp(ssp, flux_dev), B.c_telescope(sub)
        ws = torch.empty(B.rubix_workspace_bytes(records.shape[0], cs, ct), dtype=torch.uint8, device=self.device)
        if mirror_lo is not None or mirror_hi is not None:
            B.rubix_build_cube_mirrored(cp, cs, ct, R, out, mirror_lo, mirror_hi, mirror_rows, ws)
        else:
            B.rubix_build_cube(cp, cs, ct, R, out, ws)
        return ws                                           # kept alive by the caller until the stream has run

    def convolve_rows(self, rows, tel):
        B, torch = self.B, self.torch
        sub = dataclasses.replace(tel, n_x=int(rows.shape[0]), n_x_full=0, x_first=0)
        ct = B.c_telescope(sub)
        out = torch.empty_like(rows)
        ws = torch.empty(B.rubix_workspace_bytes(0, None, ct), dtype=torch.uint8, device=self.device)
        B.rubix_convolve_psf_lsf(ct, rows, out, ws)
        return out

    def upload_flux(self, ssp):
        return self.torch.from_numpy(np.ascontiguousarray(ssp.flux)).to(self.device)


def pack_records(particles, device):
    """[n, 9] fp32 tensor (pos, vel, mass, log_age, log_z) of a synth.Particles / any object with those arrays."""
    import torch
    rec = np.concatenate([particles.pos, particles.vel, particles.mass[:, None], particles.log_age[:, None],
                          particles.log_z[:, None]], axis=1).astype(np.float32)
    return torch.from_numpy(np.ascontiguousarray(rec)).to(device)


# ------------------------------------------------------------------------------------------ the sharded forward
@dataclasses.dataclass
class Slab:
    x0: int
    x1: int
    cube: object             # tensor [x1 - x0, n_y, n_c]: this rank's rows of the final cube
    bounds: np.ndarray
    n_received: int


def forward_sharded(comm, backend, records, R, ssp, tel, flux_dev=None, row_cost=None, fuse_halo=True) -> Slab:
    """SPMD: every rank calls this with ITS slice of the particle records (contiguous slices of the original arrays in rank
    order).  Returns the rank's slab of the final cube.  ``tel`` is the whole detector.  ``fuse_halo``: use the fused halo write
    (rubix_build_cube_mirrored) where the communicator lets ranks store into each other's buffers."""
    import torch
    n_x, n_y, n_c = int(tel.n_x), int(tel.n_y), int(tel.n_channels)
    rank, world = comm.rank, comm.world
    halo = (int(tel.psf_size) - 1) // 2 if int(tel.psf_size) > 0 else 0
    # 1-2  keys of my particles in the whole detector's geometry, particles per detector row (global)
    key = backend.bin(records, tel, R).to(torch.int64)
    inside = key < n_x * n_y
    rows = torch.div(key, n_y, rounding_mode="floor")
    counts = torch.bincount(rows[inside], minlength=n_x).to(torch.int64)
    counts = comm.all_reduce_sum(counts)
    # the order of summation inside a spaxel (rubix_telescope.cell_order) is decided ONCE, from the whole galaxy, as a
    # single-GPU call on it would decide: every rank then accumulates its spaxels in that order
    if int(getattr(tel, "cell_order", 0)) == 0:
        n_total = int(comm.all_reduce_sum(torch.tensor([records.shape[0]], dtype=torch.int64, device=key.device))[0].item())
        tel = dataclasses.replace(tel, cell_order=2 if n_total >= max(CELL_AUTO_MIN_N, CELL_AUTO_MEAN * n_x * n_y) else 1)
    # 3  the same partition on every rank
    bounds = partition_rows(counts.cpu().numpy(), world, min_rows=max(1, halo),
                            row_cost=float(n_y) if row_cost is None else row_cost)
    # 4  particle records to the owners of their rows, original order kept inside every message
    dest = owner_of_rows(rows, bounds)
    sends = {d: records[inside & (dest == d)] for d in range(world)}
    n_to = torch.tensor([sends[d].shape[0] for d in range(world)], dtype=torch.int64, device=records.device)
    n_from = [int(c[rank].item()) for c in comm.all_gather_counts(n_to)]
    got = comm.exchange({d: t for d, t in sends.items() if d != rank},
                        {s: (n_from[s], RECORD_FLOATS) for s in range(world) if s != rank}, records)
    got[rank] = sends[rank]
    mine = torch.cat([got[s] for s in range(world)], dim=0).contiguous()
    # 5  my raw rows, in a buffer with room for the neighbours' rows
    x0, x1 = int(bounds[rank]), int(bounds[rank + 1])
    h_lo, h_hi = (halo if rank > 0 else 0), (halo if rank < world - 1 else 0)
    n_own = x1 - x0
    buf = torch.zeros((h_lo + n_own + h_hi, n_y, n_c), dtype=getattr(backend, "dtype", torch.float32), device=records.device)
    if flux_dev is None:
        flux_dev = backend.upload_flux(ssp)
    conv = int(tel.psf_size) > 0 or int(tel.lsf_size) > 0
    # 5 + 6 fused where the ranks can store into each other's buffers (one address space / mapped peer memory): the kernels
    # that produce my boundary rows also write them into the neighbours' halos, and the exchange shrinks to a barrier
    peers = None
    if fuse_halo and conv and halo > 0 and world > 1:
        if records.is_cuda:
            torch.cuda.current_stream().synchronize()      # my buffer is zero-filled before a neighbour may store into it
        peers = comm.share(buf)
    if peers is not None:
        lo_peer = hi_peer = None
        if rank > 0:                                        # my first rows are the UPPER halo of rank - 1
            b_lo = peers[rank - 1]
            lo_peer = b_lo[b_lo.shape[0] - halo:]
        if rank < world - 1:                                # my last rows are the LOWER halo of rank + 1
            hi_peer = peers[rank + 1][0:halo]
        keep = backend.build_rows(mine, R, ssp, flux_dev, tel, x0, x1, buf[h_lo:h_lo + n_own], lo_peer, hi_peer, halo)
        if records.is_cuda:
            torch.cuda.current_stream().synchronize()
        comm.barrier()                                      # every rank's rows (and mirrors) are complete
    else:
        keep = backend.build_rows(mine, R, ssp, flux_dev, tel, x0, x1, buf[h_lo:h_lo + n_own])
    if not conv:
        if records.is_cuda:
            torch.cuda.current_stream().synchronize()
        del keep
        return Slab(x0, x1, buf, bounds, int(mine.shape[0]))
    # 6  halo exchange: my first / last `halo` rows are the neighbours' upper / lower halo
    if peers is None and halo > 0 and world > 1:
        if records.is_cuda:
            torch.cuda.current_stream().synchronize()      # the rows must be complete before a peer reads them
        sends, recvs = {}, {}
        if rank > 0:
            sends[rank - 1] = buf[h_lo:h_lo + halo]
            recvs[rank - 1] = (halo, n_y, n_c)
        if rank < world - 1:
            sends[rank + 1] = buf[h_lo + n_own - halo:h_lo + n_own]
            recvs[rank + 1] = (halo, n_y, n_c)
        halos = comm.exchange(sends, recvs, buf)
        if rank > 0:
            buf[0:h_lo].copy_(halos[rank - 1])
        if rank < world - 1:
            buf[h_lo + n_own:].copy_(halos[rank + 1])
    # 7  stencils on rows + halos; the halo rows of the result are discarded
    final = backend.convolve_rows(buf, tel)
    if records.is_cuda:
        torch.cuda.current_stream().synchronize()
    del keep
    return Slab(x0, x1, final[h_lo:h_lo + n_own].contiguous(), bounds, int(mine.shape[0]))


def slice_for_rank(n: int, rank: int, world: int):
    """Contiguous slice of the original particle arrays held by ``rank`` (rank order = original order)."""
    per = (n + world - 1) // world
    return slice(min(rank * per, n), min((rank + 1) * per, n))
