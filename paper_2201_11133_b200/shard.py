"""Host-side logic of the multi-GPU path: the hot path shards over independent windows
(gwi_infer) or over contiguous time spans of a stream (gwi_stream_*); models are replicated and no collective sits on
the data path (one rank per GPU, no inter-rank traffic during inference).  The only exchange is at the
end: timing (max over ranks), trigger counts, and -- for time shards -- the runs that touch a shard edge, which are
merged here.  No arithmetic of the network lives in this module; it is index bookkeeping, tested on CPU with gloo.
"""
from dataclasses import dataclass
from typing import List, Sequence, Tuple


def plan_windows(n_windows: int, world: int) -> List[Tuple[int, int]]:
    """Contiguous [start, end) window ranges, sizes differing by at most one, in rank order."""
    base, extra = divmod(int(n_windows), int(world))
    out, pos = [], 0
    for r in range(world):
        n = base + (1 if r < extra else 0)
        out.append((pos, pos + n))
        pos += n
    return out


@dataclass
class TimeShard:
    rank: int
    start: int          # first output sample this rank owns
    end: int            # one past the last
    warm_start: int     # first input sample it has to read: start - (R_f - 1), clipped at 0 (exact history, pin P8)
    l1_start: int       # first L1 sample it needs for the slides: warm_start - max_lag, clipped at 0 (the circular wrap
                        # of rank 0 is served by the stream tail, as in gwi_stream_prime)


def plan_time(n_samples: int, world: int, receptive_field: int, max_lag: int = 0, align: int = 1) -> List[TimeShard]:
    """Contiguous time spans, boundaries on multiples of `align`, each with the warm-up it needs in front."""
    out, pos = [], 0
    for r, (a, b) in enumerate(plan_windows((n_samples + align - 1) // align, world)):
        s, e = min(a * align, n_samples), min(b * align, n_samples)
        ws = max(0, s - (receptive_field - 1))
        out.append(TimeShard(r, s, e, ws, max(0, ws - max_lag)))
        pos = e
    assert pos == n_samples
    return out


def merge_shard_runs(shard_runs: Sequence[Sequence[Tuple[int, int]]], bounds: Sequence[Tuple[int, int]], min_len: int):
    """shard_runs[r]: ALL maximal supra-threshold runs [s, e) found inside shard r's span bounds[r] = (start, end), in
    global sample indices (min_len not yet applied; a run is cut at the span edges).  Runs that end exactly at a shard's
    end and a run that starts exactly at the next shard's start are one run of the whole stream.  Returns the merged
    runs of length >= min_len, sorted by start -- the list gwi_ensemble_triggers gives on the unsharded stream."""
    merged: List[List[int]] = []
    for r, runs in enumerate(shard_runs):
        lo, hi = bounds[r]
        for s, e in sorted(runs):
            assert lo <= s < e <= hi
            if merged and merged[-1][1] == s and s == lo and r > 0:
                merged[-1][1] = e           # continues the run that touched the previous shard's end
            else:
                merged.append([s, e])
    return [(s, e) for s, e in merged if e - s >= min_len]


def reduce_step_time(ms_local: float, dist=None) -> float:
    """Max over ranks of a per-rank device time (the bench contract); identity without a process group."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms_local)
    import torch
    t = torch.tensor([float(ms_local)], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def gather_objects(obj, dist=None):
    """All ranks' python objects on every rank (trigger lists / boundary runs are a few hundred bytes per rank)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return [obj]
    out = [None] * dist.get_world_size()
    dist.all_gather_object(out, obj)
    return out
