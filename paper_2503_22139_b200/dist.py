"""Multi-GPU plumbing: one process per GPU.  Two modes:
  replicas  every rank runs an independent replica of the step, no data-path collective (bench.py default);
  z-slabs   every rank owns a contiguous range of brick layers (slab_bounds), forward is
            collective-free, backward sums the per-Gaussian accumulators with ONE all-reduce
            (sharded_backward) between gsvox_backward_accumulate and gsvox_backward_finish.  torch.distributed is used for the rendezvous, the barriers around the timed
region and the max-over-ranks reduction of the device time.  Backend nccl on GPUs, gloo in the CPU
tests (tests/test_dist_gloo.py, world_size 2)."""
import os

import torch
import torch.distributed as dist


class Ranks:
    def __init__(self, backend=None):
        self.rank = int(os.environ.get("RANK", "0"))
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.local = int(os.environ.get("LOCAL_RANK", "0"))
        self.backend = backend or ("nccl" if torch.cuda.is_available() else "gloo")
        self.on = self.world > 1
        if self.on and not dist.is_initialized():
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            kw = {}
            if self.backend == "nccl":
                kw["device_id"] = torch.device("cuda", self.local)
            dist.init_process_group(self.backend, rank=self.rank, world_size=self.world, **kw)

    def _dev(self):
        return torch.device("cuda", self.local) if self.backend == "nccl" else torch.device("cpu")

    def barrier(self):
        if self.on:
            dist.barrier()
        if self.backend == "nccl" and torch.cuda.is_available():
            torch.cuda.synchronize()

    def max_over_ranks(self, value):
        t = torch.tensor([float(value)], dtype=torch.float64, device=self._dev())
        if self.on:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    def sum_over_ranks(self, value):
        t = torch.tensor([float(value)], dtype=torch.float64, device=self._dev())
        if self.on:
            dist.all_reduce(t, op=dist.ReduceOp.SUM)
        return float(t.item())

    def close(self):
        if self.on and dist.is_initialized():
            dist.barrier()
            dist.destroy_process_group()


def whole_job_rate(units_per_rank, ranks, ms_total, steps):
    """value = units all ranks processed / max-over-ranks time (weak scaling, replicas)."""
    ms_step = ranks.max_over_ranks(ms_total) / steps
    total_units = ranks.sum_over_ranks(units_per_rank)
    return total_units / (ms_step * 1e-3), ms_step


def slab_bounds(nbz, rank, world):
    """Balanced contiguous split of the nbz brick layers (8 voxels each) along z: rank r owns layers
    [lo, hi).  Covers 0..nbz exactly once; ranks beyond nbz get an empty slab."""
    if not (0 <= rank < world) or nbz < 0:
        raise ValueError("slab_bounds(nbz=%r, rank=%r, world=%r)" % (nbz, rank, world))
    base, extra = divmod(nbz, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def slab_bounds_by_keys(layer_keys, rank, world):
    """Contiguous split of the brick layers balanced by KEY COUNT, not by layer count: layer_keys[l] = keys whose
    brick lies in layer l (Plan.layer_keys() of an unsharded binning, or any work estimate).  Clustered inputs
    (config 5's blobs) make layers very unequal: equal-layer slabs leave most ranks idle.  Rank r owns [lo, hi);
    cut c sits at the layer boundary whose running sum is nearest to c/world of the total (ties to the left, cuts
    never move backwards), so every layer is owned exactly once, slabs stay contiguous, and equal weights reproduce slab_bounds up to rounding.
    All ranks must pass the same layer_keys."""
    nbz = len(layer_keys)
    if not (0 <= rank < world):
        raise ValueError("slab_bounds_by_keys(rank=%r, world=%r)" % (rank, world))
    total = float(sum(layer_keys))
    if nbz == 0 or total <= 0:
        return slab_bounds(nbz, rank, world)
    prefix = [0.0]
    for v in layer_keys:
        prefix.append(prefix[-1] + float(v))
    cuts = [0]
    for c in range(1, world):                      # the boundary whose prefix sum is nearest to c/world of the total
        target = total * c / world
        best = cuts[-1]
        for i in range(cuts[-1], nbz + 1):
            if abs(prefix[i] - target) < abs(prefix[best] - target):
                best = i
        cuts.append(best)
    cuts.append(nbz)
    return cuts[rank], cuts[rank + 1]


def sharded_backward(plan, weight, grad_out, ranks, grads=None, all_reduce=None):
    """a4 on this rank's slab -> sum of the [n, 9 + C] accumulators over ranks -> a5.  `all_reduce`
    defaults to torch.distributed.all_reduce (NCCL over NVLink/NVSwitch: 24 MB at config 4)."""
    ch = int(weight.shape[1])
    plan.backward_accumulate(weight, grad_out)
    if ranks.on:
        (all_reduce or dist.all_reduce)(plan.accumulators(ch))
    return plan.backward_finish(ch, grads=grads)


def batch_bounds(batch, rank, world):
    """The 8(f) operators (combine, warp, projector, rasterizer) are independent per projection of a batch:
    rank r takes projections [lo, hi) of the B, no data-path collective in forward; in backward only the
    gradients of the SHARED parameters (Gaussians, I_ref) are summed over ranks (all_reduce_grads)."""
    return slab_bounds(batch, rank, world)


def all_reduce_grads(tensors, ranks, all_reduce=None):
    """Sum per-rank partial gradients of shared parameters in place (one call per tensor; NCCL on GPUs)."""
    if ranks.on:
        for t in tensors:
            (all_reduce or dist.all_reduce)(t)
    return tensors
