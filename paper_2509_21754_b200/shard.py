"""Multi-GPU plumbing: one process per GPU, torch.distributed (NCCL on GPUs; gloo in the CPU tests).

Two ways the path spreads over ranks; neither touches a pixel here -- all arithmetic of
the method stays in the CUDA kernels behind include/fitrig.h:

* independent problems (stacks, fields, frequency channels; tiles and fields are independent, PAPER.md:122,
  209; R19): `split_range` hands every rank a contiguous share; there is NO data-path collective, only the
  barrier and the max-over-ranks of the device time (`max_over_ranks`).
* ONE image over several GPUs: horizontal shards of whole tile rows (`row_shards`).  The only coupling is
  the three global scalars of the method -- M and per unit the mean and standard deviation of
  the tile matrix (Eq. 8) -- exchanged in ONE all-gather of 2 + 2U doubles per rank
  (`ShardedContext.tlisi`; the frequency branch adds a second one of 3 doubles for the statistics of eta, which
  can only be formed once the global M is known), then the candidate lists are gathered and put in (unit, tile row, tile col)
  order (`gather_candidates`, `merge_candidates`: index bookkeeping only).
"""
from __future__ import annotations

from typing import List, Optional, Sequence, Tuple

import numpy as np

from .binding import CANDIDATE_DTYPE, Context


def split_range(n: int, world: int, rank: int) -> Tuple[int, int]:
    """Contiguous, balanced share [lo, hi) of n independent problems for `rank` of `world`."""
    if world < 1 or not (0 <= rank < world) or n < 0:
        raise ValueError("need world >= 1, 0 <= rank < world, n >= 0")
    return (rank * n) // world, ((rank + 1) * n) // world


def row_shards(H: int, tile: int, world: int) -> List[Tuple[int, int]]:
    """Image rows [r0, r1) of each shard: whole tile rows (r0 a multiple of tile), balanced to one tile row.
    The last shard takes the partial bottom tile row, if any (R5).  Shards may be empty when world > Ty."""
    if H < 1 or tile < 1 or world < 1:
        raise ValueError("need H, tile, world >= 1")
    Ty = -(-H // tile)
    out = []
    for r in range(world):
        t0, t1 = split_range(Ty, world, r)
        out.append((min(H, t0 * tile), min(H, t1 * tile)))
    return out


def _dist():
    import torch.distributed as dist
    return dist


def all_gather_vectors(v, group=None):
    """[n] tensor on every rank -> [world, n] tensor (same device and dtype), rank order.  The one exchange
    step of the sharded path; works over NCCL (CUDA tensors) and gloo (CPU tensors)."""
    import torch
    dist = _dist()
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return v.reshape(1, -1).clone()
    world = dist.get_world_size(group)
    out = torch.empty(world * v.numel(), dtype=v.dtype, device=v.device)  # flat: gloo insists on it
    dist.all_gather_into_tensor(out, v.contiguous().reshape(-1), group=group)
    return out.reshape(world, v.numel())


def max_over_ranks(value: float, device="cpu", group=None) -> float:
    """MAX all-reduce of one float (bench.py: device time of the slowest rank)."""
    import torch
    dist = _dist()
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())


def gather_candidates(local: np.ndarray, device="cpu", group=None) -> List[np.ndarray]:
    """Every rank's candidate list (structured arrays of CANDIDATE_DTYPE) on every rank, rank order."""
    import torch
    dist = _dist()
    local = np.ascontiguousarray(local, dtype=CANDIDATE_DTYPE)
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return [local.copy()]
    world = dist.get_world_size(group)
    counts = all_gather_vectors(torch.tensor([len(local)], dtype=torch.int64, device=device), group).reshape(-1)
    cap = int(counts.max().item())
    buf = torch.zeros((max(cap, 1), 4), dtype=torch.int32, device=device)  # 16-byte records as 4 x int32
    if len(local):
        buf[: len(local)] = torch.from_numpy(local.view(np.int32).reshape(-1, 4)).to(device)
    allb = all_gather_vectors(buf.reshape(-1), group).reshape(world, max(cap, 1), 4).cpu().numpy()
    return [np.ascontiguousarray(allb[r, : int(counts[r].item())]).reshape(-1).view(CANDIDATE_DTYPE).copy()
            for r in range(world)]


def merge_candidates(per_shard: Sequence[np.ndarray]) -> np.ndarray:
    """Shard lists (each ascending in (unit, tile row, tile col), shards in increasing row order) -> one list in
    the library's order guarantee: ascending (unit, tile row, tile col).  Shards own disjoint, increasing
    tile rows, so a stable sort by unit of the concatenation is the merge."""
    if not len(per_shard):
        return np.zeros(0, dtype=CANDIDATE_DTYPE)
    cat = np.concatenate([np.asarray(c, dtype=CANDIDATE_DTYPE) for c in per_shard])
    return cat[np.argsort(cat["snapshot"], kind="stable")]


def shard_host_rows(h_snapshots: Sequence, r0: int, r1: int) -> List:
    """Rows [r0, r1) of every host snapshot ([H, W] torch tensors or numpy arrays), as views: what ONE rank streams of
    an image that lives whole in (pinned) host memory.  Rows of a row-major image are contiguous, so each view is one
    contiguous block that starts r0 * W elements into its snapshot -- index bookkeeping only, nothing is copied."""
    out = []
    for s in h_snapshots:
        if s.ndim != 2 or not (0 <= r0 < r1 <= s.shape[0]):
            raise ValueError(f"rows [{r0}, {r1}) of a snapshot of shape {tuple(s.shape)}")
        v = s[r0:r1]
        contiguous = v.is_contiguous() if hasattr(v, "is_contiguous") else v.flags["C_CONTIGUOUS"]
        if not contiguous:
            raise ValueError("host snapshots must be row-major and contiguous")
        out.append(v)
    return out


class ShardedContext:
    """This rank's horizontal shard of ONE H x W image stack (image branch).

        sc = ShardedContext(H, W, L, rank, world, device=local_rank)
        sc.tlisi(d_stack_rows)            # [L, r1 - r0, W] CUDA tensor: this rank's rows of every snapshot
        cands, n = sc.detect(tau)         # this shard's candidates, y in image rows
        everyone = sc.gather(cands)       # all candidates in (unit, tile row, tile col) order, on every rank

    For an image that lives in host memory (BASELINE.json configs[3]; "sharding strips across G GPUs
    multiplies host-to-device bandwidth"), `sc.stream(h_snapshots)` takes the WHOLE host snapshots and copies only this
    rank's rows [r0, r1) of each through fitrig_stream: every rank moves H_shard * W * L * 4 bytes over its own PCIe
    link, 1 / world of the image, and the exchange that follows is the same 2 + 2U doubles.
    """

    def __init__(self, H: int, W: int, n_snapshots: int, rank: int, world: int, group=None, **params):
        tile = int(params.get("tile", 0)) or 32
        self.rank, self.world, self.group = rank, world, group
        self.rows = row_shards(H, tile, world)
        self.r0, self.r1 = self.rows[rank]
        if self.r1 <= self.r0:
            raise ValueError(f"rank {rank} of {world} has no tile row of a {H}-row image (tile {tile})")
        self.ctx = Context(self.r1 - self.r0, W, n_snapshots, row_offset=self.r0, **params)
        self.units = self.ctx.units
        self.device = int(params.get("device", 0))
        self._vec = None

    def _exchange(self, vec, stream):
        """All-gather of `vec` (written on `stream`) -> [world, n], safe to read on `stream`: the collective runs on
        torch's current stream, so the two streams are ordered against each other on both sides."""
        import torch
        cur = torch.cuda.current_stream(vec.device) if vec.is_cuda else None
        lib_stream = None
        if cur is not None and stream is not None:
            lib_stream = stream if hasattr(stream, "cuda_stream") else torch.cuda.ExternalStream(int(stream), device=vec.device)
            if lib_stream.cuda_stream != cur.cuda_stream:
                cur.wait_stream(lib_stream)  # the export kernel has written vec
            else:
                lib_stream = None
        allv = all_gather_vectors(vec, self.group)
        if lib_stream is not None:
            lib_stream.wait_stream(cur)  # the import kernel may not read allv before the collective has delivered it
        return allv

    def tlisi(self, d_stack_rows, d_tlisi=None, stream=None) -> None:
        self.ctx.tlisi(d_stack_rows, None, stream)
        self._globalise(d_stack_rows.device, d_tlisi, stream)

    def stream(self, h_snapshots: Sequence, d_tlisi=None, stream=None) -> None:
        """h_snapshots: the L WHOLE host snapshots [H, W] (pinned for overlap), the same list on every rank; this rank
        streams only its rows of each (`shard_host_rows`), then the shards exchange M and the statistics as in
        `tlisi`.  d_tlisi (device, [U, Ty_shard, Tx]) receives this shard's tLISI under the global M."""
        import torch
        self.ctx.stream(shard_host_rows(h_snapshots, self.r0, self.r1), None, stream)
        self._globalise(torch.device("cuda", self.device), d_tlisi, stream)

    def _globalise(self, device, d_tlisi, stream) -> None:
        """The exchange step: provisional shard map -> the map under the global M, mu, sigma (and eta's statistics)."""
        import torch
        if self._vec is None:
            self._vec = torch.empty(2 + 2 * self.units, dtype=torch.float64, device=device)
            self._vec_eta = torch.empty(3, dtype=torch.float64, device=device)
        self.ctx.shard_export(self._vec, stream)
        allv = self._exchange(self._vec, stream)
        self.ctx.shard_import(allv, allv.shape[0], d_tlisi, stream)
        self._all = allv  # keep alive until the kernel has read it
        if self.ctx.branch == 1:  # eta scales with 1 / M^2: its statistics need a second, 3-double exchange
            self.ctx.shard_export_eta(self._vec_eta, stream)
            alle = self._exchange(self._vec_eta, stream)
            self.ctx.shard_import_eta(alle, alle.shape[0], stream)
            self._all_eta = alle

    def detect(self, sigma_threshold: float, capacity: int = 1 << 16, stream=None):
        return self.ctx.detect(sigma_threshold, capacity, stream)

    def gather(self, local_cands: np.ndarray, device="cpu") -> np.ndarray:
        return merge_candidates(gather_candidates(local_cands, device, self.group))

    def close(self):
        self.ctx.close()

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()
