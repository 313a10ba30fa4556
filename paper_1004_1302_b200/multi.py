"""Multi-GPU additive render: particle shards + one sum-reduction of the raw-S partial images.

This is the paper's own parallel decomposition (every process renders its share of
the particles into a full-size image, the partial images are combined by a collective
reduction), legal because E_p = A_p makes the line-of-sight sum order-independent
(PAPER.md:75).  One process per GPU; every rank
  1. renders its particle shard with SPLOTCH_RAW_SUM (S_c, not 1 - exp(-S_c)),
  2. takes part in ONE all-reduce(sum, fp32) of the H*W*3 image (NCCL over NVLink/NVSwitch),
  3. applies the output map once (splotch_normalize).
There is no other exchange step.  The absorb mode does not shard by particle chunk (front-to-back
compositing is associative but not commutative): it runs as independent replicas only.

Host logic only: the render and the output map run in libsplotch_b200.so.  `combine_partials`
takes the collective and the output map as callables so that the world-size-2 gloo tests can
drive the same code path on CPU tensors.
"""
from __future__ import annotations

from typing import Callable, Optional, Tuple


def shard_bounds(n: int, world: int, rank: int) -> Tuple[int, int]:
    """[start, stop) of rank's contiguous particle chunk: equal chunks, the first n % world one longer."""
    if world < 1 or not (0 <= rank < world) or n < 0:
        raise ValueError(f"bad shard request n={n} world={world} rank={rank}")
    base, rem = divmod(n, world)
    start = rank * base + min(rank, rem)
    return start, start + base + (1 if rank < rem else 0)


def shard_workload(w, world: int, rank: int):
    """Rank's contiguous slice of a workloads.Workload-like object (arrays are views, not copies)."""
    import copy
    s, e = shard_bounds(int(w.n), world, rank)
    sh = copy.copy(w)
    for k in ("x", "y", "z", "r", "I", "colval"):
        setattr(sh, k, getattr(w, k)[s:e])
    sh.type = None if w.type is None else w.type[s:e]
    vec = getattr(w, "vec", None)           # optional (n, 3) vector colouring follows its particles
    if vec is not None:
        sh.vec = vec[s:e]
    sh.n = e - s
    return sh


def combine_partials(partial, all_reduce: Callable, output_map: Optional[Callable]):
    """partial: this rank's raw-S image (modified in place).  all_reduce(t) sums t over the ranks in
    place; output_map(t) applies out = 1 - exp(-S) in place (None keeps raw S)."""
    all_reduce(partial)
    if output_map is not None:
        output_map(partial)
    return partial


class ShardedScene:
    """A particle shard resident on this rank's GPU + the collective that finishes the image."""

    def __init__(self, w_shard, device: str, group=None):
        import torch.distributed as dist
        from .scene import Scene
        if int(w_shard.mode) != 0:
            raise ValueError("particle sharding is defined for the additive mode only (absorb: replicas only)")
        self.scene = Scene(w_shard, device)
        self.group = group
        self._dist = dist

    def render(self, cam=None, raw: bool = False, out=None, check: bool = True):
        from . import binding as B
        dist = self._dist
        img = self.scene.render(cam, raw=True, out=out, check=check)
        # the collective runs whenever a process group exists, also a group of one rank (there it is the identity): the
        # one-GPU test then executes the very call sequence of the N-GPU job
        sharded = dist.is_available() and dist.is_initialized()
        return combine_partials(
            img,
            (lambda t: dist.all_reduce(t, op=dist.ReduceOp.SUM, group=self.group)) if sharded else (lambda t: None),
            None if raw else (lambda t: B.splotch_normalize(t, t, t.numel())))
